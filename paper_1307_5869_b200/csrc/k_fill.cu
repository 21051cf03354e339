// k_fill.cu -- write-peak probe: 128-bit streaming stores of a register constant.
// The bench measures the HBM write roofline with it in the same run as the generators.
#include "k_common.cuh"

namespace prand {
namespace {

__global__ void __launch_bounds__(256)
fill_u32_kernel(uint32_t *__restrict__ out, uint64_t n_vec, uint64_t n_words, uint32_t value)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint4 v = make_uint4(value, value, value, value);
    uint4 *o = reinterpret_cast<uint4 *>(out);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) __stcs(o + i, v);
    // ragged tail (< 4 words)
    if (blockIdx.x == 0 && threadIdx.x < (n_words & 3)) out[n_vec * 4 + threadIdx.x] = value;
}

}  // namespace

cudaError_t fill_u32(cudaStream_t stream, uint32_t *out, uint64_t n_words, uint32_t value, LaunchInfo *li)
{
    const uint64_t n_vec = n_words / 4;
    uint64_t blocks = ceil_div_u64(n_vec ? n_vec : 1, 256);
    const uint64_t cap = (uint64_t)sm_count() * 16;   // grid-stride: a few CTAs per SM, many stores in flight each
    if (blocks > cap) blocks = cap;
    fill_u32_kernel<<<(unsigned)blocks, 256, 0, stream>>>(out, n_vec, n_words, value);
    li->kernel = "fill_u32";
    li->launches = 1;
    return cudaGetLastError();
}

}  // namespace prand
