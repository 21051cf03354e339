// k_lfsr113.cu -- LFSR113 jump and generation kernels.
//
// four shift-register sequences x_n = x_{n-p} + x_{n-p+q} (mod 2) (eq. 7), each
// emitting u_n = sum_{i=1..32} x_{ns+i-1} 2^-i (eq. 8), (p,q,s) = (31,6,18), (29,2,2), (28,13,7),
// (25,3,13); the output is the XOR of the four words.  With z holding bits x_{ns}..x_{ns+31} MSB
// first, one output step of a component is
//     z' = ((z & top_p) << s) ^ (((z << q) ^ z) >> (p - s)).
// Jump-ahead: n steps are a GF(2)-linear map of the word, stored by columns (LfsrOp).
// State layout (SoA): z[c * n_streams + s], c = 0..3.
#include "k_common.cuh"
#include "../../include/prand_device.cuh"

namespace prand {
namespace {

// the component step, the combined step and the GF(2) skip are the device-callable API's (one definition)
using prand_dev::tausworthe;
using prand_dev::lfsr113_step;
using prand_dev::lfsr113_apply_bits;

__global__ void __launch_bounds__(256)
lfsr113_jump_kernel(const uint32_t *__restrict__ base, const uint32_t *st_in,
                    uint32_t *st_out, uint64_t ns, const LfsrOp *__restrict__ ops,
                    uint64_t idx0, uint64_t idx_stride)
{
    uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    uint32_t z[4];
    for (int c = 0; c < 4; c++) z[c] = base ? base[c] : st_in[c * ns + s];
    lfsr113_apply_bits(ops, idx0 + s * idx_stride, z);
    for (int c = 0; c < 4; c++) st_out[c * ns + s] = z[c];
}

// ---- the paper's own jump algorithm (section 5.3) as an alternate --------------------
// By eq. 9 the sequence decimated by k = 2^e, y_l = x_{kl}, obeys the recurrence (7) itself.  A "table"
// starts from p consecutive bits, extends them to 2p - 1 with (7) (the row x_{2^n p} .. x_{2^n (2p-1)} of the
// paper) and keeps every second bit: after n rounds it holds x_0, x_{2^n}, ..., x_{(p-1) 2^n}, and bit s of
// it is x_{s 2^n}, the first bit of the output word 2^n steps ahead (eq. 8).  Bit i of that word comes from
// the table started at x_i: 32 tables per component, 128 per stream -- "constructed independently using
// different threads": one warp per stream, lane = start bit, each lane runs its four components; the new
// state words are assembled with a warp ballot.  A jump by E 2^b outputs is the succession of the jumps
// 2^(i + b) over the set bits i of E.  Words are kept MSB first (bit 63 - k of a 64-bit register = x_k).
template <int P, int Q, int S> __device__ __forceinline__ uint32_t tausworthe_table_bit(uint32_t z, int lane, unsigned n);

__device__ __forceinline__ uint64_t keep_even_msb_first(uint64_t y)
{
    y &= 0xAAAAAAAAAAAAAAAAull;                           // indices 0, 2, 4, ... (MSB first) = odd bit positions
    y = (y | (y << 1)) & 0xCCCCCCCCCCCCCCCCull;
    y = (y | (y << 2)) & 0xF0F0F0F0F0F0F0F0ull;
    y = (y | (y << 4)) & 0xFF00FF00FF00FF00ull;
    y = (y | (y << 8)) & 0xFFFF0000FFFF0000ull;
    y = (y | (y << 16)) & 0xFFFFFFFF00000000ull;
    return y;
}
// (v, valid): the top `valid` bits of v are sequence bits; extend to `target` bits with eq. 7
template <int P, int Q> __device__ __forceinline__ uint64_t taus_extend(uint64_t v, int valid, int target)
{
    while (valid < target) {
        int g = (P - Q < target - valid) ? P - Q : target - valid;
        uint64_t t = (v >> P) ^ (v >> (P - Q));          // bit index i holds x_{i-P} ^ x_{i-P+Q}
        uint64_t m = (~0ull >> valid) & ~((valid + g >= 64) ? 0ull : (~0ull >> (valid + g)));
        v |= t & m;
        valid += g;
    }
    return v;
}
template <int P, int Q, int S> __device__ __forceinline__ uint32_t tausworthe_table_bit(uint32_t z, int lane, unsigned n)
{
    constexpr uint32_t top_p = 0xFFFFFFFFu << (32 - P);
    constexpr uint64_t top_p64 = ~0ull << (64 - P);
    uint64_t y = taus_extend<P, Q>((uint64_t)(z & top_p) << 32, P, 64) << lane;    // the table's p start bits x_lane ..
    y &= top_p64;
    for (unsigned r = 0; r < n; r++) y = keep_even_msb_first(taus_extend<P, Q>(y, P, 2 * P - 1)) & top_p64;
    return (uint32_t)(y >> (63 - S)) & 1u;
}

constexpr int TABLE_WARPS = 4;
__global__ void __launch_bounds__(32 * TABLE_WARPS)
lfsr113_table_jump_kernel(const uint32_t *__restrict__ base, const uint32_t *st_in, uint32_t *st_out, uint64_t ns,
                          uint64_t mant, unsigned log2, uint64_t idx0, uint64_t idx_stride)
{
    const uint64_t s = (uint64_t)blockIdx.x * TABLE_WARPS + (threadIdx.x >> 5);
    if (s >= ns) return;                                    // whole warp
    const int lane = threadIdx.x & 31;
    uint32_t z[4];
    for (int c = 0; c < 4; c++) z[c] = base ? base[c] : st_in[c * ns + s];
    uint64_t e = (idx0 + s * idx_stride) * mant;            // the launcher guarantees no overflow
    for (unsigned i = 0; e != 0; i++, e >>= 1) {
        if (!(e & 1)) continue;
        const unsigned n = i + log2;                        // jump 2^n outputs
        const uint32_t b0 = tausworthe_table_bit<31, 6, 18>(z[0], lane, n);
        const uint32_t b1 = tausworthe_table_bit<29, 2, 2>(z[1], lane, n);
        const uint32_t b2 = tausworthe_table_bit<28, 13, 7>(z[2], lane, n);
        const uint32_t b3 = tausworthe_table_bit<25, 3, 13>(z[3], lane, n);
        // lane i holds bit x_{s 2^n + i} = bit 31 - i of the new word
        z[0] = __brev(__ballot_sync(0xFFFFFFFFu, b0));
        z[1] = __brev(__ballot_sync(0xFFFFFFFFu, b1));
        z[2] = __brev(__ballot_sync(0xFFFFFFFFu, b2));
        z[3] = __brev(__ballot_sync(0xFFFFFFFFu, b3));
    }
    if (lane < 4) st_out[lane * ns + s] = lane == 0 ? z[0] : lane == 1 ? z[1] : lane == 2 ? z[2] : z[3];
}

// ---- bit-stream form of one component (hot path) -------------------------------------------------
// Successive output words of a component overlap: word n is bits x_{ns}..x_{ns+31} of ONE bit
// sequence, so an output consumes only s fresh bits (18 + 2 + 7 + 13 = 40 for the four components)
// while the word form recomputes 4 x 5 shift/logic operations.  Here the sequence is kept as 32-bit
// words W_j = x_{32j}..x_{32j+31} (MSB first) and extended a whole word at a time with eq. 9
// (PAPER.md:363-368): x_n = x_{n-Kp} + x_{n-Kp+Kq} for K = 2^e.  A word needs K(p-q) >= 32 so that
// every operand bit is already known: K = 2 for components 1, 2, 4 and K = 4 for component 3.
// Each new word is two funnel shifts and one XOR; output n is one funnel shift at bit offset
// n*s mod 32, a compile-time constant when 32 outputs are unrolled (after 32 outputs the offset is
// back to 0 and the sequence has advanced exactly s words).  ~9.75 ALU operations per output
// instead of 22.
template <int R> __device__ __forceinline__ uint32_t funnel(uint32_t first, uint32_t second)
{
    // 32 bits starting R bits into the 64-bit string first:second (MSB first)
    if constexpr (R == 0) return first;
    else return __funnelshift_l(second, first, R);
}

template <int P, int Q, int S> struct TausBits {
    static constexpr int K = (2 * (P - Q) >= 32) ? 2 : 4;
    static constexpr int H = K;                                     // ring of history words
    static constexpr int R1 = 32 * K - K * P, R2 = R1 + K * Q;      // bit offsets of the two taps from word j-K
    static_assert(K * (P - Q) >= 32 && R1 >= 0 && R2 + 32 <= 32 * K, "eq. 9 taps must lie in known words");
    uint32_t w[H];                                                  // word j lives in w[j % H]

    __host__ __device__ static constexpr int need(int n) { return (n * S + 31) / 32; }  // last word output n touches
    __host__ __device__ static constexpr int upto(int n) { return need(n) > H - 1 ? need(n) : H - 1; }

    // (v, valid): the top `valid` bits of v are sequence bits; extend to `target` bits with eq. 7
    __device__ static __forceinline__ uint64_t extend(uint64_t v, int valid, int target)
    {
        while (valid < target) {
            int g = (P - Q < target - valid) ? P - Q : target - valid;
            uint64_t t = (v >> P) ^ (v >> (P - Q));                 // bit index i holds x_{i-P} ^ x_{i-P+Q}
            uint64_t m = (~0ull >> valid) & ~((valid + g >= 64) ? 0ull : (~0ull >> (valid + g)));
            v |= t & m;
            valid += g;
        }
        return v;
    }
    // from the state word z (top P bits significant): words 0..H-1 of the sequence starting at z
    __device__ __forceinline__ void load(uint32_t z)
    {
        constexpr uint32_t top_p = 0xFFFFFFFFu << (32 - P);
        uint64_t v = extend((uint64_t)(z & top_p) << 32, P, 64);
        w[0] = (uint32_t)(v >> 32);
        w[1] = (uint32_t)v;
#pragma unroll
        for (int j = 2; j < H; j++) w[j] = (uint32_t)extend((uint64_t)w[j - 1] << 32, 32, 64);
    }
    template <int J> __device__ __forceinline__ void gen()          // word J from words J-K..J-1
    {
        constexpr int A1 = J - K + (R1 >> 5), A2 = J - K + (R2 >> 5);
        uint32_t t1 = funnel<(R1 & 31)>(w[A1 % H], w[(A1 + 1) % H]);
        uint32_t t2 = funnel<(R2 & 31)>(w[A2 % H], w[(A2 + 1) % H]);
        w[J % H] = t1 ^ t2;
    }
    template <int J0, int J1> __device__ __forceinline__ void gen_range()
    {
        if constexpr (J0 <= J1) { gen<J0>(); gen_range<J0 + 1, J1>(); }
    }
    // output N = 1..32 of the current block (step-then-output: output N is the word at bit N*S)
    template <int N> __device__ __forceinline__ uint32_t output()
    {
        gen_range<upto(N - 1) + 1, upto(N)>();
        constexpr int a = (N * S) / 32, r = (N * S) % 32;
        return funnel<r>(w[a % H], w[(a + 1) % H]);
    }
    // after output 32 the sequence has advanced S words: make word S the new word 0
    __device__ __forceinline__ void next_block()
    {
        gen_range<upto(32) + 1, S + H - 1>();
        uint32_t t[H];
#pragma unroll
        for (int i = 0; i < H; i++) t[i] = w[(S + i) % H];
#pragma unroll
        for (int i = 0; i < H; i++) w[i] = t[i];
    }
    __device__ __forceinline__ uint32_t state() const { return w[0]; }   // all 32 bits are sequence bits
};

template <int V> struct LfsrBits {
    TausBits<31, 6, 18> c1[V];
    TausBits<29, 2, 2> c2[V];
    TausBits<28, 13, 7> c3[V];
    TausBits<25, 3, 13> c4[V];
};

template <int V, int DT, int N>
__device__ __forceinline__ void lfsr113_emit_rows(LfsrBits<V> &b, typename OutElem<DT>::type *&p, uint64_t ns)
{
    if constexpr (N <= 32) {
        typename OutElem<DT>::type r[V];
#pragma unroll
        for (int v = 0; v < V; v++)
            r[v] = convert<DT>(b.c1[v].template output<N>() ^ b.c2[v].template output<N>() ^
                               b.c3[v].template output<N>() ^ b.c4[v].template output<N>());
        store_vec<V>(p, r);
        p += ns;
        lfsr113_emit_rows<V, DT, N + 1>(b, p, ns);
    }
}

// One thread owns V adjacent streams (V = 4: one 128-bit store per row for u32/f32, two for f64)
// and one row chunk (blockIdx.y).  Threads of a warp own adjacent stream groups, so a warp writes
// 32*V consecutive elements of a row per step.  Rows go out in blocks of 32 in the bit-stream form;
// a ragged tail (< 32 rows) uses the word form.
constexpr int GEN_THREADS = 128;

template <int V, int DT>
__global__ void __launch_bounds__(GEN_THREADS)
lfsr113_gen_kernel(const uint32_t *st_in, uint32_t *st_out,
                   typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n,
                   uint64_t chunk_len, const LfsrOp *__restrict__ chunk_ops)
{
    typedef typename OutElem<DT>::type T;
    const uint64_t sg = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t s0 = sg * V;
    if (s0 >= ns) return;
    const uint32_t c = blockIdx.y;

    uint32_t z[V][4];
#pragma unroll
    for (int k = 0; k < 4; k++) {
        if constexpr (V == 4) {
            uint4 t = *reinterpret_cast<const uint4 *>(st_in + k * ns + s0);
            z[0][k] = t.x; z[1][k] = t.y; z[2][k] = t.z; z[3][k] = t.w;
        } else {
#pragma unroll
            for (int v = 0; v < V; v++) z[v][k] = st_in[k * ns + s0 + v];
        }
    }
    if (c != 0) {
#pragma unroll
        for (int v = 0; v < V; v++) lfsr113_apply_bits(chunk_ops + (c - 1), 1, z[v]);   // operator of c * chunk_len
    }
    const uint64_t row0 = (uint64_t)c * chunk_len;
    const uint64_t rows = (row0 + chunk_len < n) ? chunk_len : n - row0;
    T *p = out + row0 * ns + s0;
    const uint64_t blocks32 = rows / 32;
    if (blocks32) {
        LfsrBits<V> b;
#pragma unroll
        for (int v = 0; v < V; v++) { b.c1[v].load(z[v][0]); b.c2[v].load(z[v][1]); b.c3[v].load(z[v][2]); b.c4[v].load(z[v][3]); }
#pragma unroll 1
        for (uint64_t blk = 0; blk < blocks32; blk++) {
            lfsr113_emit_rows<V, DT, 1>(b, p, ns);
#pragma unroll
            for (int v = 0; v < V; v++) { b.c1[v].next_block(); b.c2[v].next_block(); b.c3[v].next_block(); b.c4[v].next_block(); }
        }
#pragma unroll
        for (int v = 0; v < V; v++) {
            z[v][0] = b.c1[v].state(); z[v][1] = b.c2[v].state(); z[v][2] = b.c3[v].state(); z[v][3] = b.c4[v].state();
        }
    }
#pragma unroll 1
    for (uint64_t i = blocks32 * 32; i < rows; i++) {
        T r[V];
#pragma unroll
        for (int v = 0; v < V; v++) r[v] = convert<DT>(lfsr113_step(z[v]));
        store_vec<V>(p, r);
        p += ns;
    }
    if (c == gridDim.y - 1) {
#pragma unroll
        for (int k = 0; k < 4; k++)
#pragma unroll
            for (int v = 0; v < V; v++) st_out[k * ns + s0 + v] = z[v][k];
    }
}

// ---- sections of a single sequence (prand_generate_seq_*; Table 5) ----------------------
// The array layout is PRAND's contiguous one, out[c * sec_len + i].  One thread per section (lane = section); a
// warp collects a block of 32 rows of its 32 sections in a shared-memory tile (pitch 33: conflict-free both ways)
// and writes it section by section: 16 bytes per lane, the lanes of a section storing its 32 consecutive numbers
// as one contiguous run (128 bytes for u32 / f32, 256 for f64).  No scratch array, no transposition pass.
template <int DT, int N>
__device__ __forceinline__ void lfsr113_emit_tile(LfsrBits<1> &b, typename OutElem<DT>::type *t)
{
    if constexpr (N <= 32) {
        t[N - 1] = convert<DT>(b.c1[0].template output<N>() ^ b.c2[0].template output<N>() ^
                               b.c3[0].template output<N>() ^ b.c4[0].template output<N>());
        lfsr113_emit_tile<DT, N + 1>(b, t);
    }
}

template <int DT>
__global__ void __launch_bounds__(GEN_THREADS)
lfsr113_seq_kernel(const uint32_t *st_in, typename OutElem<DT>::type *__restrict__ out, uint64_t n_sections,
                   uint64_t sec_len, uint64_t length)
{
    typedef typename OutElem<DT>::type T;
    constexpr int PITCH = 33;
    constexpr int EPL = 16 / (int)sizeof(T);               // elements per lane and store (4 or 2)
    constexpr int LPS = 32 / EPL;                          // lanes per section
    constexpr int SPP = 32 / LPS;                          // sections per pass
    __shared__ T tile_all[GEN_THREADS / 32][32 * PITCH];
    T *tile = tile_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const uint64_t warp_sec0 = (uint64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u);
    if (warp_sec0 >= n_sections) return;                   // whole warp
    const uint64_t sec = warp_sec0 + lane < n_sections ? warp_sec0 + lane : n_sections - 1;
    LfsrBits<1> b;
    b.c1[0].load(st_in[0 * n_sections + sec]);
    b.c2[0].load(st_in[1 * n_sections + sec]);
    b.c3[0].load(st_in[2 * n_sections + sec]);
    b.c4[0].load(st_in[3 * n_sections + sec]);
    const uint64_t last = n_sections - 1, last_rows = length - last * sec_len;
    const bool whole = warp_sec0 + 32 <= n_sections && (warp_sec0 + 32 <= last || last_rows == sec_len);
    const int sub = lane / LPS, piece = lane % LPS;
    T *dst0 = out + (warp_sec0 + sub) * sec_len + EPL * piece;
    const T *tsrc = tile + sub * PITCH + EPL * piece;
#pragma unroll 1
    for (uint64_t i0 = 0; i0 < sec_len; i0 += 32) {        // (sec_len is a multiple of 32)
        lfsr113_emit_tile<DT, 1>(b, tile + lane * PITCH);
        b.c1[0].next_block(); b.c2[0].next_block(); b.c3[0].next_block(); b.c4[0].next_block();
        __syncwarp();
        T *d = dst0 + i0;
#pragma unroll
        for (int k = 0; k < 32 / SPP; k++) {
            T v[EPL];
#pragma unroll
            for (int e = 0; e < EPL; e++) v[e] = tsrc[k * SPP * PITCH + e];
            if (whole) {
                store_vec<EPL>(d, v);
            } else {
                const uint64_t c = warp_sec0 + SPP * k + sub;
                if (c < n_sections) {
                    const uint64_t rows = c == last ? last_rows : sec_len, row = i0 + EPL * piece;
#pragma unroll
                    for (int e = 0; e < EPL; e++)
                        if (row + e < rows) store1(d + e, v[e]);
                }
            }
            d += (uint64_t)SPP * sec_len;
        }
        __syncwarp();
    }
}

template <int V, int DT>
cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type T;
    dim3 grid((unsigned)ceil_div_u64(a.n_streams / V, GEN_THREADS), (unsigned)a.n_chunks);
    lfsr113_gen_kernel<V, DT><<<grid, GEN_THREADS, 0, stream>>>(
        (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (T *)a.out, a.n_streams, a.n, a.chunk_len,
        (const LfsrOp *)a.chunk_ops);
    return cudaGetLastError();
}

template <int DT> cudaError_t dispatch_v(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    // 128-bit stores need 4 adjacent streams per thread and 16-byte aligned rows.
    bool vec = (a.n_streams % 4 == 0) && ((uintptr_t)a.out % 16 == 0) && ((uintptr_t)a.st_in % 16 == 0) &&
               !lfsr113_narrow(a.n_streams, a.n, a.dtype, sm_count());
    li->launches = 1;
    if (vec) { li->kernel = "lfsr113_gen<V=4>"; return launch_gen<4, DT>(stream, a); }
    li->kernel = "lfsr113_gen<V=1>";
    return launch_gen<1, DT>(stream, a);
}

}  // namespace

cudaError_t lfsr113_jump(cudaStream_t stream, const JumpArgs &a, LaunchInfo *li)
{
    unsigned blocks = (unsigned)ceil_div_u64(a.n_streams, 256);
    lfsr113_jump_kernel<<<blocks, 256, 0, stream>>>((const uint32_t *)a.base, (const uint32_t *)a.st_in,
                                                    (uint32_t *)a.st_out, a.n_streams,
                                                    (const LfsrOp *)a.ops, a.idx0, a.idx_stride);
    li->kernel = "lfsr113_jump";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t lfsr113_seq(cudaStream_t stream, const void *st_in, void *out, int dtype, uint64_t n_sections, uint64_t sec_len,
                        uint64_t length, LaunchInfo *li)
{
    const unsigned blocks = (unsigned)ceil_div_u64(ceil_div_u64(n_sections, 32) * 32, GEN_THREADS);
    switch (dtype) {
    case DT_U32: lfsr113_seq_kernel<DT_U32><<<blocks, GEN_THREADS, 0, stream>>>((const uint32_t *)st_in, (uint32_t *)out, n_sections, sec_len, length); break;
    case DT_F32: lfsr113_seq_kernel<DT_F32><<<blocks, GEN_THREADS, 0, stream>>>((const uint32_t *)st_in, (float *)out, n_sections, sec_len, length); break;
    default: lfsr113_seq_kernel<DT_F64><<<blocks, GEN_THREADS, 0, stream>>>((const uint32_t *)st_in, (double *)out, n_sections, sec_len, length); break;
    }
    li->kernel = "lfsr113_seq";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t lfsr113_table_jump(cudaStream_t stream, const JumpArgs &a, uint64_t mant, unsigned log2, LaunchInfo *li)
{
    unsigned blocks = (unsigned)ceil_div_u64(a.n_streams, TABLE_WARPS);
    lfsr113_table_jump_kernel<<<blocks, 32 * TABLE_WARPS, 0, stream>>>((const uint32_t *)a.base, (const uint32_t *)a.st_in,
                                                                      (uint32_t *)a.st_out, a.n_streams, mant, log2,
                                                                      a.idx0, a.idx_stride);
    li->kernel = "lfsr113_table_jump";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t lfsr113_generate(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    switch (a.dtype) {
    case DT_U32: return dispatch_v<DT_U32>(stream, a, li);
    case DT_F32: return dispatch_v<DT_F32>(stream, a, li);
    default: return dispatch_v<DT_F64>(stream, a, li);
    }
}

}  // namespace prand
