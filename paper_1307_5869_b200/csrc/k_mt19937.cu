// k_mt19937.cu -- MT19937 jump-polynomial application and generation kernels
// (SURVEY.md 8(a) a1, a2, a5, a7, a8).
//
// MT19937 (algorithm of the paper's ref. [2]) is linear over F_2, Y_{n+1} = A Y_n;
// jump-ahead is A^v Y_0 = g_v(A) Y_0 = a_k Y_{k-1} + ... + a_1 Y_0, k = 19937 (eq. 10), with
// g_v(x) = x^v mod phi(x).  Recurrence (ref. [2] parameters, reading T1):
//   x_{i+624} = x_{i+397} ^ (y >> 1) ^ (y odd ? 0x9908B0DF : 0),  y = (x_i & 0x80000000) | (x_{i+1} & 0x7FFFFFFF),
// output number P = temper(x_{P+624}); the state at position P is the window x_P..x_{P+623}.
// State layout: [stream][624] u32 (one stream's window is contiguous: a warp loads it coalesced).
#include "k_common.cuh"

namespace prand {
namespace {

constexpr int NW = 624, MW = 397, DEG = 19937;

__device__ __forceinline__ uint32_t mt_recur(uint32_t xi, uint32_t xi1, uint32_t xim)
{
    uint32_t y = (xi & 0x80000000u) | (xi1 & 0x7FFFFFFFu);
    return xim ^ (y >> 1) ^ ((0u - (y & 1u)) & 0x9908B0DFu);
}
__device__ __forceinline__ uint32_t mt_temper(uint32_t y)
{
    y ^= y >> 11;
    y ^= (y << 7) & 0x9D2C5680u;
    y ^= (y << 15) & 0xEFC60000u;
    y ^= y >> 18;
    return y;
}

// ---- eq. 10 in correlation form -----------------------------------------------------------------
// One CTA per destination stream.  The source window is extended to x_0..x_{19937+623} in shared
// memory (227 independent words per round), then output word j is the XOR of x_{i+j}
// over the set coefficients a_i of g_v.
constexpr int APPLY_THREADS = 256;
constexpr int APPLY_XWORDS = DEG + NW;
constexpr size_t APPLY_SMEM = (size_t)(APPLY_XWORDS + NW) * sizeof(uint32_t);

__global__ void __launch_bounds__(APPLY_THREADS)
mt19937_apply_kernel(const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                     uint64_t src_back, const MtOp *__restrict__ op)
{
    extern __shared__ uint32_t smem[];
    uint32_t *x = smem;                    // APPLY_XWORDS
    uint32_t *poly = smem + APPLY_XWORDS;  // NW
    const int tid = threadIdx.x;
    const uint64_t dst = dst0 + blockIdx.x;
    const uint32_t *src = st_src + (dst - src_back) * NW;
    for (int j = tid; j < NW; j += APPLY_THREADS) {
        x[j] = src[j];
        poly[j] = op->w[j];
    }
    __syncthreads();
    for (int r0 = 0; r0 < DEG; r0 += 227) {
        int k = r0 + tid;
        if (tid < 227 && k < DEG) x[NW + k] = mt_recur(x[k], x[k + 1], x[k + MW]);
        __syncthreads();
    }
    // thread t accumulates output words t, t+256, t+512 (the last only for t < 112)
    uint32_t acc0 = 0, acc1 = 0, acc2 = 0;
    const uint32_t *x0 = x + tid, *x1 = x + tid + 256;
    const uint32_t *x2 = x + (tid + 512 < NW ? tid + 512 : 0);
    for (int wi = 0; wi < NW; wi++) {
        uint32_t pw = poly[wi];            // uniform over the CTA
        while (pw) {
            int i = wi * 32 + (__ffs(pw) - 1);
            pw &= pw - 1;
            acc0 ^= x0[i];
            acc1 ^= x1[i];
            acc2 ^= x2[i];
        }
    }
    uint32_t *d = st_dst + dst * NW;
    d[tid] = tid == 0 ? (acc0 & 0x80000000u) : acc0;   // only the top bit of word 0 is state (T2)
    d[tid + 256] = acc1;
    if (tid + 512 < NW) d[tid + 512] = acc2;
}

// ---- generation ----------------------------------------------------------------------------------
// CTA = G warps; warp w owns stream s0 + w with its 624-word window as a circular buffer in shared
// memory; lane l produces x_{P+624+l}, 32 new words per round (the recurrence reaches back 227 >= 32
// words, so a round's 32 words are independent).  Rounds of all G warps are transposed through a
// [32][G] tile so that each output row segment out[i*ns + s0 .. s0+G) is written contiguously.
template <int G, int DT>
__global__ void __launch_bounds__(G * 32)
mt19937_gen_kernel(const uint32_t *st_in, uint32_t *st_out,
                   typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n)
{
    typedef typename OutElem<DT>::type T;
    constexpr int PITCH = G + 1;
    extern __shared__ uint32_t smem[];
    uint32_t *xs = smem;                       // [G][NW]
    uint32_t *tile = smem + G * NW;            // [2][32][PITCH]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t s0 = (uint64_t)blockIdx.x * G;
    const uint64_t s = s0 + warp;
    const bool live = s < ns;
    uint32_t *x = xs + warp * NW;
    if (live)
        for (int j = lane; j < NW; j += 32) x[j] = st_in[s * NW + j];
    __syncwarp();
    int h = 0;                                 // slot of x_P
    int buf = 0;
    for (uint64_t t0 = 0; t0 < n; t0 += 32, buf ^= 1) {
        const int rem = (n - t0 < 32) ? (int)(n - t0) : 32;
        uint32_t *tl = tile + buf * 32 * PITCH;
        if (live) {
            int a = h + lane;      if (a >= NW) a -= NW;
            int b = a + 1;         if (b >= NW) b -= NW;
            int m = a + MW;        if (m >= NW) m -= NW;
            uint32_t nw = mt_recur(x[a], x[b], x[m]);
            __syncwarp();
            if (lane < rem) x[a] = nw;
            __syncwarp();
            tl[lane * PITCH + warp] = mt_temper(nw);
            h += rem; if (h >= NW) h -= NW;
        }
        __syncthreads();
        {
            const int row = threadIdx.x / G, col = threadIdx.x % G;
            if (row < rem && s0 + col < ns)
                store1(out + (t0 + row) * ns + s0 + col, convert<DT>(tl[row * PITCH + col]));
        }
    }
    if (live) {
        __syncwarp();
        for (int j = lane; j < NW; j += 32) {
            int a = h + j; if (a >= NW) a -= NW;
            uint32_t v = x[a];
            st_out[s * NW + j] = v;
        }
    }
}

template <int G, int DT> cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type T;
    size_t smem = (size_t)(G * NW + 2 * 32 * (G + 1)) * sizeof(uint32_t);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(mt19937_gen_kernel<G, DT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    unsigned blocks = (unsigned)ceil_div_u64(a.n_streams, G);
    mt19937_gen_kernel<G, DT><<<blocks, G * 32, smem, stream>>>((const uint32_t *)a.st_in, (uint32_t *)a.st_out,
                                                              (T *)a.out, a.n_streams, a.n);
    return cudaGetLastError();
}

template <int G> cudaError_t dispatch_dt(cudaStream_t stream, const GenArgs &a)
{
    switch (a.dtype) {
    case DT_U32: return launch_gen<G, DT_U32>(stream, a);
    case DT_F32: return launch_gen<G, DT_F32>(stream, a);
    default: return launch_gen<G, DT_F64>(stream, a);
    }
}

}  // namespace

cudaError_t mt19937_apply(cudaStream_t stream, const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                          uint64_t count, uint64_t src_back, const MtOp *d_op, LaunchInfo *li)
{
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(mt19937_apply_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)APPLY_SMEM);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    li->kernel = "mt19937_apply";
    li->launches = 0;
    // grid.x is limited to 2^31-1 blocks; streams beyond that would not fit device memory anyway
    if (count == 0) return cudaSuccess;
    mt19937_apply_kernel<<<(unsigned)count, APPLY_THREADS, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t mt19937_generate(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    li->launches = 1;
    // few streams: small CTAs so that more SMs get work; many streams: full 128-byte row segments
    if (a.n_streams >= 32ull * 2 * (uint64_t)sm_count()) {
        li->kernel = "mt19937_gen<G=32>";
        return dispatch_dt<32>(stream, a);
    }
    li->kernel = "mt19937_gen<G=8>";
    return dispatch_dt<8>(stream, a);
}

}  // namespace prand
