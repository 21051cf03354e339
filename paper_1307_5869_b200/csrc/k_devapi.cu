// k_devapi.cu -- a kernel written against the device-callable API of include/prand_device.cuh
// (PAPER.md:410, 437-446): one thread per stream calls next_*() in a plain loop and
// writes the canonical layout out[i * n_streams + s].  It is the library's own example / self-test of
// that header (tests compare it with the oracle and with the bulk kernels); it is not a fast path.
#include "k_common.cuh"
#include "../../include/prand_device.cuh"

namespace prand {
namespace {

template <int GEN, int DT>
__global__ void __launch_bounds__(64)
devapi_kernel(void *state, typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    prand_dev::Gen<GEN> g;
    g.load(state, ns, s);
    for (uint64_t i = 0; i < n; i++) {
        if constexpr (DT == DT_U32) out[i * ns + s] = g.next_u32();
        else if constexpr (DT == DT_F32) out[i * ns + s] = g.next_f32();
        else out[i * ns + s] = g.next_f64();
    }
    g.store(state, ns, s);
}

template <int GEN> cudaError_t launch(cudaStream_t stream, void *state, void *out, uint64_t ns, uint64_t n, int dtype)
{
    const unsigned blocks = (unsigned)ceil_div_u64(ns, 64);
    if (dtype == DT_U32) devapi_kernel<GEN, DT_U32><<<blocks, 64, 0, stream>>>(state, (uint32_t *)out, ns, n);
    else if (dtype == DT_F32) devapi_kernel<GEN, DT_F32><<<blocks, 64, 0, stream>>>(state, (float *)out, ns, n);
    else devapi_kernel<GEN, DT_F64><<<blocks, 64, 0, stream>>>(state, (double *)out, ns, n);
    return cudaGetLastError();
}

}  // namespace

cudaError_t devapi_generate(cudaStream_t stream, int gen, void *state, void *out, uint64_t ns, uint64_t n,
                            int dtype, LaunchInfo *li)
{
    li->kernel = "devapi_example";
    li->launches = 1;
    switch (gen) {
    case PRAND_LFSR113: return launch<PRAND_LFSR113>(stream, state, out, ns, n, dtype);
    case PRAND_MRG32K3A: return launch<PRAND_MRG32K3A>(stream, state, out, ns, n, dtype);
    case PRAND_MT19937: return launch<PRAND_MT19937>(stream, state, out, ns, n, dtype);
    case PRAND_GM19: return launch<PRAND_GM19>(stream, state, out, ns, n, dtype);
    case PRAND_GM29: return launch<PRAND_GM29>(stream, state, out, ns, n, dtype);
    case PRAND_GM31: return launch<PRAND_GM31>(stream, state, out, ns, n, dtype);
    case PRAND_GM55: return launch<PRAND_GM55>(stream, state, out, ns, n, dtype);
    case PRAND_GM61: return launch<PRAND_GM61>(stream, state, out, ns, n, dtype);
    case PRAND_GQ58_1: return launch<PRAND_GQ58_1>(stream, state, out, ns, n, dtype);
    case PRAND_GQ58_3: return launch<PRAND_GQ58_3>(stream, state, out, ns, n, dtype);
    case PRAND_GQ58_4: return launch<PRAND_GQ58_4>(stream, state, out, ns, n, dtype);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace prand
