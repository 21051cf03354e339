// k_fill.cu -- write-peak probe: 128-bit streaming stores of a register constant.
// The bench measures the HBM write roofline with it in the same run as the generators.
#include "k_common.cuh"

namespace prand {
namespace {

// One 128-bit store per thread, CTAs in launch order: the write front stays compact (a few MB) because new CTAs are
// handed out in index order as old ones retire.  Measured on B200 over 8 GiB: 7.58 TB/s, against 6.3-7.0 TB/s for a
// grid-stride loop of the same stores (4-32 CTAs per SM; threads drift apart and the fronts scatter over DRAM pages),
// 7.50 / 7.21 / 6.93 / 6.33 TB/s for CTAs that own contiguous 64 KB / 256 KB / 1 MB / 4 MB pieces, 6.4 TB/s for
// cp.async.bulk stores of 32 KB pieces, 7.40 TB/s for cudaMemsetAsync; cache hints (.cs, .cg, .wt, L1::no_allocate)
// and 256-bit stores change nothing.  This is the write roofline the HBM rows of bench.py are divided by.
__global__ void __launch_bounds__(256)
fill_u32_kernel(uint32_t *__restrict__ out, uint64_t n_vec, uint64_t n_words, uint32_t value)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_vec) __stcs(reinterpret_cast<uint4 *>(out) + i, make_uint4(value, value, value, value));
    // ragged tail (< 4 words)
    if (blockIdx.x == 0 && threadIdx.x < (n_words & 3)) out[n_vec * 4 + threadIdx.x] = value;
}

// Sections of a single sequence (prand_generate_seq_*): the bulk kernels fill the family of sections
// in the interleaved layout tmp[i * S + c]; PRAND's array layout is out[c * L + i].
// 32 x 32 tiles through shared memory, both sides coalesced.
template <class E>
__global__ void __launch_bounds__(256)
transpose_sections_kernel(const E *__restrict__ tmp, E *__restrict__ out, uint64_t S, uint64_t L, uint64_t length)
{
    __shared__ E tile[32][33];
    const uint64_t i0 = (uint64_t)blockIdx.x * 32, c0 = (uint64_t)blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const uint64_t i = i0 + r, c = c0 + tx;
        if (i < L && c < S) tile[r][tx] = tmp[i * S + c];
    }
    __syncthreads();
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const uint64_t c = c0 + r, i = i0 + tx;
        if (c < S && i < L && c * L + i < length) __stcs(out + c * L + i, tile[tx][r]);
    }
}

}  // namespace

cudaError_t transpose_sections(cudaStream_t stream, const void *tmp, void *out, uint64_t n_sections,
                               uint64_t sec_len, uint64_t length, int elem_bytes, LaunchInfo *li)
{
    dim3 grid((unsigned)ceil_div_u64(sec_len, 32), (unsigned)ceil_div_u64(n_sections, 32));
    if (elem_bytes == 8)
        transpose_sections_kernel<uint64_t><<<grid, 256, 0, stream>>>((const uint64_t *)tmp, (uint64_t *)out,
                                                                      n_sections, sec_len, length);
    else
        transpose_sections_kernel<uint32_t><<<grid, 256, 0, stream>>>((const uint32_t *)tmp, (uint32_t *)out,
                                                                      n_sections, sec_len, length);
    li->kernel = "transpose_sections";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t fill_u32(cudaStream_t stream, uint32_t *out, uint64_t n_words, uint32_t value, LaunchInfo *li)
{
    const uint64_t n_vec = n_words / 4;
    const uint64_t blocks = ceil_div_u64(n_vec ? n_vec : 1, 256);
    if (blocks > 0x7FFFFFFFull) return cudaErrorInvalidValue;      // 2^31 CTAs x 4 KiB = 8 TiB
    fill_u32_kernel<<<(unsigned)blocks, 256, 0, stream>>>(out, n_vec, n_words, value);
    li->kernel = "fill_u32";
    li->launches = 1;
    return cudaGetLastError();
}

}  // namespace prand
