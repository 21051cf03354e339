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
#include "k_common.cuh"

namespace prand {
namespace {

constexpr int NW = 624, MW = 397, DEG = 19937;

__device__ __forceinline__ uint32_t mt_recur(uint32_t xi, uint32_t xi1, uint32_t xim)
{
    uint32_t y = (xi & 0x80000000u) | (xi1 & 0x7FFFFFFFu);
    return xim ^ (y >> 1) ^ ((0u - (y & 1u)) & 0x9908B0DFu);
}

// ---- eq. 10 in correlation form -----------------------------------------------------------------
// One CTA per destination stream.  The source window is extended to x_0..x_{19937+623} in shared
// memory (227 independent words per round), then output word j is the XOR of x_{i+j}
// over the set coefficients a_i of g_v.  The coefficients are expanded, 2048 at a time, into a list of
// set positions in shared memory, so that the accumulation loop has no bit scan and runs eight
// positions (24 independent shared loads per thread) at a time; the list is padded with a position
// whose words are zero.
constexpr int APPLY_XWORDS = DEG + NW;                      // 20561
constexpr int APPLY_ZERO = APPLY_XWORDS;                    // x[APPLY_ZERO .. +APPLY_ZPAD) = 0
constexpr int APPLY_ZPAD = 771;                             // >= 768, makes the list 16-byte aligned
constexpr int APPLY_CHUNK = 64;                             // polynomial words per expansion
constexpr int APPLY_LIST = APPLY_CHUNK * 32 + 8;            // positions (u16) incl. padding
constexpr size_t APPLY_SMEM = (size_t)(APPLY_XWORDS + APPLY_ZPAD) * sizeof(uint32_t) + APPLY_LIST * sizeof(uint16_t) + 16;

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
    constexpr int APPLY_THREADS = NT, NOUT = NW / SPLIT, NO = (NOUT + NT - 1) / NT;
    static_assert(NW % SPLIT == 0, "SPLIT must divide 624");
    const int out0 = (int)(blockIdx.x % SPLIT) * NOUT;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *x = smem;                                                      // APPLY_XWORDS + APPLY_ZPAD
    uint16_t *list = reinterpret_cast<uint16_t *>(smem + APPLY_XWORDS + APPLY_ZPAD);  // APPLY_LIST
    int *meta = reinterpret_cast<int *>(list + APPLY_LIST);                  // [0] warp-0 total, [1] count
    const int tid = threadIdx.x;
    const uint64_t dst = dst0 + blockIdx.x / SPLIT;
    const uint32_t *src = st_src + (dst - src_back) * NW;
    for (int j = tid; j < NW; j += APPLY_THREADS) x[j] = src[j];
    for (int j = tid; j < APPLY_ZPAD; j += APPLY_THREADS) x[APPLY_ZERO + j] = 0;
    __syncthreads();
    constexpr int EXT = NT < NW - MW ? NT : NW - MW;       // at most 227 new words are independent
    for (int r0 = 0; r0 < DEG; r0 += EXT) {
        int k = r0 + tid;
        if (tid < EXT && k < DEG) x[NW + k] = mt_recur(x[k], x[k + 1], x[k + MW]);
        __syncthreads();
    }
    // thread t accumulates output words t, t + NT, ... (those below 624)
    uint32_t acc[NO];
    const uint32_t *xo[NO];
#pragma unroll
    for (int o = 0; o < NO; o++) {
        acc[o] = 0;
        xo[o] = x + (tid + NT * o < NOUT ? out0 + tid + NT * o : 0);
    }
    for (int c0 = 0; c0 < NW; c0 += APPLY_CHUNK) {
        // expand polynomial words c0 .. c0+63 (threads 0..63, two warps) into the list of set positions
        if (tid < APPLY_CHUNK) {
            const int wi = c0 + tid;
            uint32_t pw = wi < NW ? __ldg(&op->w[wi]) : 0u;
            const int cnt = __popc(pw);
            int incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
                if ((tid & 31) >= d) incl += v;
            }
            if (tid == 31) meta[0] = incl;
            __syncwarp();
            asm volatile("bar.sync 1, 64;" ::: "memory");
            int pos = incl - cnt + (tid >= 32 ? meta[0] : 0);
            if (tid == APPLY_CHUNK - 1) meta[1] = pos + cnt;
            while (pw) {
                list[pos++] = (uint16_t)(wi * 32 + (__ffs(pw) - 1));
                pw &= pw - 1;
            }
        }
        __syncthreads();
        const int n = meta[1];
        if (tid < 8) list[n + tid] = (uint16_t)APPLY_ZERO;
        __syncthreads();
        for (int k = 0; k < n; k += 8) {
            const uint4 q = *reinterpret_cast<const uint4 *>(list + k);      // eight positions, uniform
            const uint32_t ii[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int h = 0; h < 4; h++) {
                const int ia = ii[h] & 0xFFFF, ib = ii[h] >> 16;
#pragma unroll
                for (int o = 0; o < NO; o++) acc[o] ^= xo[o][ia] ^ xo[o][ib];
            }
        }
        __syncthreads();
    }
    uint32_t *d = st_dst + dst * NW;
#pragma unroll
    for (int o = 0; o < NO; o++) {
        const int j = out0 + tid + NT * o;
        if (tid + NT * o < NOUT) d[j] = j == 0 ? (acc[o] & 0x80000000u) : acc[o];   // only the top bit of word 0 is state (T2)
    }
}

// Throughput form of the same application (many destination streams).  Thread t accumulates the four
// consecutive output words 4t .. 4t+3.  For the 32 coefficients of one polynomial word pw (positions
// 32 wi + b) they read x[32 wi + 4t + b + c], c < 4: a window of 35 consecutive words, loaded as nine
// aligned 16-byte shared loads into registers; bit b of pw (the same for all threads) then predicates
// four register XORs.  36 words loaded per 64 XORs on average instead of one load per XOR.
constexpr int APPLYW_THREADS = 160;                         // 156 active in the accumulation

__global__ void __launch_bounds__(APPLYW_THREADS)
mt19937_apply_win_kernel(const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                         uint64_t src_back, const MtOp *__restrict__ op)
{
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *x = smem;                                    // APPLY_XWORDS + APPLY_ZPAD
    const int tid = threadIdx.x;
    const uint64_t dst = dst0 + blockIdx.x;
    const uint32_t *src = st_src + (dst - src_back) * NW;
    for (int j = tid; j < NW; j += APPLYW_THREADS) x[j] = src[j];
    for (int j = tid; j < APPLY_ZPAD; j += APPLYW_THREADS) x[APPLY_ZERO + j] = 0;
    __syncthreads();
    for (int r0 = 0; r0 < DEG; r0 += APPLYW_THREADS) {
        int k = r0 + tid;
        if (k < DEG) x[NW + k] = mt_recur(x[k], x[k + 1], x[k + MW]);
        __syncthreads();
    }
    if (tid >= NW / 4) return;
    uint32_t acc[4][4] = {};                               // four interleaved sets: independent XOR chains
    const uint4 *xw = reinterpret_cast<const uint4 *>(x) + tid;   // window of wi starts at xw[8 wi]
    // two register windows in ping-pong: the nine loads of the next polynomial word are issued before
    // the 128 predicated XORs of the current one
    uint4 wa[9], wb[9];
    auto load_win = [&](uint4 (&w)[9], int wi) {
#pragma unroll
        for (int q = 0; q < 9; q++) w[q] = xw[8 * wi + q];
    };
    auto accumulate = [&](const uint4 (&w)[9], uint32_t pw) {
        uint32_t v[36];
#pragma unroll
        for (int q = 0; q < 9; q++) { v[4 * q] = w[q].x; v[4 * q + 1] = w[q].y; v[4 * q + 2] = w[q].z; v[4 * q + 3] = w[q].w; }
#pragma unroll
        for (int b = 0; b < 32; b++) {
            if (pw & (1u << b)) {
                acc[b & 3][0] ^= v[b]; acc[b & 3][1] ^= v[b + 1]; acc[b & 3][2] ^= v[b + 2]; acc[b & 3][3] ^= v[b + 3];
            }
        }
    };
    load_win(wa, 0);
    uint32_t pw0 = __ldg(&op->w[0]), pw1 = __ldg(&op->w[1]);
#pragma unroll 1
    for (int wi = 0; wi < NW; wi += 2) {
        load_win(wb, wi + 1);
        const uint32_t p0 = pw0, p1 = pw1;
        if (wi + 2 < NW) { pw0 = __ldg(&op->w[wi + 2]); pw1 = __ldg(&op->w[wi + 3]); }
        accumulate(wa, p0);
        load_win(wa, wi + 2 < NW ? wi + 2 : wi);
        accumulate(wb, p1);
    }
    uint32_t *d = st_dst + dst * NW + 4 * tid;
    uint32_t r[4];
#pragma unroll
    for (int c = 0; c < 4; c++) r[c] = acc[0][c] ^ acc[1][c] ^ acc[2][c] ^ acc[3][c];
    *reinterpret_cast<uint4 *>(d) = make_uint4(tid == 0 ? (r[0] & 0x80000000u) : r[0], r[1], r[2], r[3]);
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
__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
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
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
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
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
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

}  // namespace

cudaError_t mt19937_apply(cudaStream_t stream, const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                          uint64_t count, uint64_t src_back, const MtOp *d_op, LaunchInfo *li)
{
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(mt19937_apply_kernel<256, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)APPLY_SMEM);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(mt19937_apply_kernel<640, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)APPLY_SMEM);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(mt19937_apply_kernel<160, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)APPLY_SMEM);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(mt19937_apply_win_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)APPLY_SMEM);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    li->kernel = "mt19937_apply";
    li->launches = 0;
    // grid.x is limited to 2^31-1 blocks; streams beyond that would not fit device memory anyway
    if (count == 0) return cudaSuccess;
    // fewer CTAs than SMs: the launch is as long as one application
    if (src_back != 0 && 4 * count <= 2 * (uint64_t)sm_count())
        mt19937_apply_kernel<160, 4><<<(unsigned)(4 * count), 160, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    else if (count <= (uint64_t)sm_count())
        mt19937_apply_kernel<640, 1><<<(unsigned)count, 640, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    else if (std::getenv("PRAND_MT_APPLY_LIST"))             // test hook: the position-list kernel at any size
        mt19937_apply_kernel<256, 1><<<(unsigned)count, 256, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    else
        mt19937_apply_win_kernel<<<(unsigned)count, APPLYW_THREADS, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t mt19937_generate(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    li->launches = 1;
    // a thread's byte offset inside a row block must fit 32 bits (wave of 208 rows, 8-byte elements)
    if (a.n_streams > ((1ull << 32) / (208 * 8)) - 8) return cudaErrorInvalidValue;
    // Kernel choice by stream count (measured on B200): 32 streams per CTA need >= ~128
    // CTAs; below that 8 streams per CTA; below ~1000 streams 4 per CTA in sector-sharing cluster pairs.
    int cfg = a.n_streams >= 4096 ? 0 : a.n_streams >= 1024 ? 1 : 2;
    if (const char *env = std::getenv("PRAND_MT_CFG")) cfg = std::atoi(env);   // test hook: force a variant
    switch (cfg) {
    case 0: li->kernel = "mt19937_bgen<S=32>"; return dispatch_bdt<0>(stream, a);
    case 1: li->kernel = "mt19937_gen<S=8,T=104>"; return dispatch_dt<8, 104, 2, 0, false>(stream, a);
    default: li->kernel = "mt19937_gen<S=4,T=208,pair>"; return dispatch_dt<4, 208, 1, 6, true>(stream, a);
    }
}

}  // namespace prand
