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

namespace prand {
namespace {

template <int P, int Q, int S> __device__ __forceinline__ uint32_t tausworthe(uint32_t z)
{
    constexpr uint32_t kept = (0xFFFFFFFFu << (32 - P)) << S;   // (z & top_p) << s == (z << s) & kept
    uint32_t b = ((z << Q) ^ z) >> (P - S);
    return ((z << S) & kept) ^ b;
}

__device__ __forceinline__ uint32_t lfsr113_step(uint32_t (&z)[4])
{
    z[0] = tausworthe<31, 6, 18>(z[0]);
    z[1] = tausworthe<29, 2, 2>(z[1]);
    z[2] = tausworthe<28, 13, 7>(z[2]);
    z[3] = tausworthe<25, 3, 13>(z[3]);
    return z[0] ^ z[1] ^ z[2] ^ z[3];
}

__device__ __forceinline__ uint32_t gf2_matvec(const uint32_t *__restrict__ col, uint32_t z)
{
    uint32_t r = 0;
#pragma unroll 8
    for (int j = 0; j < 32; j++) r ^= (0u - ((z >> j) & 1u)) & __ldg(col + j);
    return r;
}

__device__ __forceinline__ void lfsr113_apply_bits(const LfsrOp *__restrict__ ops, uint64_t idx,
                                                   uint32_t (&z)[4])
{
    for (int lev = 0; idx != 0; lev++, idx >>= 1)
        if (idx & 1)
            for (int c = 0; c < 4; c++) z[c] = gf2_matvec(ops[lev].col[c], z[c]);
}

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

// One thread owns V adjacent streams (V = 4: one 128-bit store per row for u32/f32, two for f64)
// and one row chunk.  Threads of a warp own adjacent stream groups, so a warp writes 32*V
// consecutive elements of a row per step.
template <int V, int DT>
__global__ void __launch_bounds__(256)
lfsr113_gen_kernel(const uint32_t *st_in, uint32_t *st_out,
                   typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n,
                   uint64_t chunk_len, uint64_t n_chunks, const LfsrOp *__restrict__ chunk_ops)
{
    typedef typename OutElem<DT>::type T;
    const uint64_t groups = ns / V;
    const uint64_t vid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vid >= groups * n_chunks) return;
    const uint64_t c = vid / groups, sg = vid - c * groups;
    const uint64_t s0 = sg * V;

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
    const uint64_t row0 = c * chunk_len;
    const uint64_t row1 = (row0 + chunk_len < n) ? row0 + chunk_len : n;
    T *p = out + row0 * ns + s0;
#pragma unroll 4
    for (uint64_t i = row0; i < row1; i++) {
        T r[V];
#pragma unroll
        for (int v = 0; v < V; v++) r[v] = convert<DT>(lfsr113_step(z[v]));
        store_vec<V>(p, r);
        p += ns;
    }
    if (c == n_chunks - 1) {
#pragma unroll
        for (int k = 0; k < 4; k++)
#pragma unroll
            for (int v = 0; v < V; v++) st_out[k * ns + s0 + v] = z[v][k];
    }
}

template <int V, int DT>
cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type T;
    uint64_t threads = (a.n_streams / V) * a.n_chunks;
    unsigned blocks = (unsigned)ceil_div_u64(threads, 256);
    lfsr113_gen_kernel<V, DT><<<blocks, 256, 0, stream>>>(
        (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (T *)a.out, a.n_streams, a.n, a.chunk_len,
        a.n_chunks, (const LfsrOp *)a.chunk_ops);
    return cudaGetLastError();
}

template <int DT> cudaError_t dispatch_v(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    // 128-bit stores need 4 adjacent streams per thread and 16-byte aligned rows.
    bool vec = (a.n_streams % 4 == 0) && ((uintptr_t)a.out % 16 == 0) && ((uintptr_t)a.st_in % 16 == 0);
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

cudaError_t lfsr113_generate(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    switch (a.dtype) {
    case DT_U32: return dispatch_v<DT_U32>(stream, a, li);
    case DT_F32: return dispatch_v<DT_F32>(stream, a, li);
    default: return dispatch_v<DT_F64>(stream, a, li);
    }
}

}  // namespace prand
