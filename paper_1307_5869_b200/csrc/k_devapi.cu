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

// Stream initialisation ON THE DEVICE (rng_dev_init_sequence_ / rng_dev_skipahead_):
// thread s loads the base stream, skips s * dist ahead with the operator table of prand_device_ops and
// generates n numbers of stream s -- the block-split family of prand_init without prand_init.
template <int GEN, int DT>
__global__ void __launch_bounds__(64)
devapi_init_kernel(const void *base, const void *ops, typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    prand_dev::Gen<GEN> g;
    g.load(base, 1, 0);
    if constexpr (GEN == PRAND_LFSR113) g.skipahead(static_cast<const prand_lfsr113_op *>(ops), s);
    else if constexpr (GEN == PRAND_MRG32K3A) g.skipahead(static_cast<const prand_mrg32k3a_op *>(ops), s);
    else g.skipahead(static_cast<const prand_gm_op *>(ops), s);
    for (uint64_t i = 0; i < n; i++) {
        if constexpr (DT == DT_U32) out[i * ns + s] = g.next_u32();
        else if constexpr (DT == DT_F32) out[i * ns + s] = g.next_f32();
        else out[i * ns + s] = g.next_f64();
    }
}

// MT19937: one CTA per stream.  The CTA-cooperative skip-ahead applies the level polynomials of the set
// bits of s to the window in shared memory, then warp 0 drives the warp-cooperative generator on it.
constexpr int MT_INIT_THREADS = 256;
constexpr size_t MT_INIT_SMEM = prand_dev::MT_SKIP_WORK_BYTES + 16 + prand_dev::MT_N * sizeof(uint32_t);

template <int DT>
__global__ void __launch_bounds__(MT_INIT_THREADS)
devapi_mt_init_kernel(const uint32_t *base, const prand_mt19937_op *ops, typename OutElem<DT>::type *__restrict__ out,
                      uint64_t ns, uint64_t n)
{
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *win = smem + (prand_dev::MT_SKIP_WORK_BYTES + 15) / 16 * 4;
    const uint64_t s = blockIdx.x;
    for (int j = threadIdx.x; j < prand_dev::MT_N; j += MT_INIT_THREADS) win[j] = base[j];
    __syncthreads();
    uint64_t idx = s;
    for (int lev = 0; idx != 0; lev++, idx >>= 1)
        if (idx & 1) prand_dev::mt19937_skipahead_cta<MT_INIT_THREADS>(smem, ops + lev, win, win);
    if (threadIdx.x >= 32) return;
    prand_dev::Gen<PRAND_MT19937> g;
    g.attach(win);
    const int lane = threadIdx.x;
    for (uint64_t i = 0; i < n; i += 32) {
        if constexpr (DT == DT_U32) { const uint32_t v = g.next_u32(); if (i + lane < n) out[(i + lane) * ns + s] = v; }
        else if constexpr (DT == DT_F32) { const float v = g.next_f32(); if (i + lane < n) out[(i + lane) * ns + s] = v; }
        else { const double v = g.next_f64(); if (i + lane < n) out[(i + lane) * ns + s] = v; }
    }
}

template <int GEN> cudaError_t launch_init(cudaStream_t stream, const void *base, const void *ops, void *out, uint64_t ns,
                                           uint64_t n, int dtype)
{
    if constexpr (GEN == PRAND_MT19937) {
        cudaError_t e = cudaSuccess;
#define PRAND_MT_INIT(DTV, TV)                                                                                      \
        e = cudaFuncSetAttribute(devapi_mt_init_kernel<DTV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MT_INIT_SMEM); \
        if (e != cudaSuccess) return e;                                                                             \
        devapi_mt_init_kernel<DTV><<<(unsigned)ns, MT_INIT_THREADS, MT_INIT_SMEM, stream>>>(                        \
            (const uint32_t *)base, (const prand_mt19937_op *)ops, (TV *)out, ns, n);
        if (dtype == DT_U32) { PRAND_MT_INIT(DT_U32, uint32_t) }
        else if (dtype == DT_F32) { PRAND_MT_INIT(DT_F32, float) }
        else { PRAND_MT_INIT(DT_F64, double) }
#undef PRAND_MT_INIT
        return cudaGetLastError();
    } else {
        const unsigned blocks = (unsigned)ceil_div_u64(ns, 64);
        if (dtype == DT_U32) devapi_init_kernel<GEN, DT_U32><<<blocks, 64, 0, stream>>>(base, ops, (uint32_t *)out, ns, n);
        else if (dtype == DT_F32) devapi_init_kernel<GEN, DT_F32><<<blocks, 64, 0, stream>>>(base, ops, (float *)out, ns, n);
        else devapi_init_kernel<GEN, DT_F64><<<blocks, 64, 0, stream>>>(base, ops, (double *)out, ns, n);
        return cudaGetLastError();
    }
}

// MT19937 on the library's state: one warp per stream on a shared-memory window (warp-cooperative generator)
template <int DT>
__global__ void __launch_bounds__(128)
devapi_mt_kernel(void *state, typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n)
{
    __shared__ uint32_t windows[4][prand_dev::MT_N];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint64_t s = (uint64_t)blockIdx.x * 4 + w;
    if (s >= ns) return;                                   // whole warp
    prand_dev::Gen<PRAND_MT19937> g;
    g.attach(windows[w]);
    g.load(state, ns, s);
    for (uint64_t i = 0; i < n; i += 32) {
        // a partial last batch: only the first n - i words may advance the stream, so it runs one number at a time
        if (i + 32 <= n) {
            if constexpr (DT == DT_U32) out[(i + lane) * ns + s] = g.next_u32();
            else if constexpr (DT == DT_F32) out[(i + lane) * ns + s] = g.next_f32();
            else out[(i + lane) * ns + s] = g.next_f64();
        } else {
            for (uint64_t k = i; k < n; k++) {
                const uint32_t v = g.next_one();
                if (lane == 0) {
                    if constexpr (DT == DT_U32) out[k * ns + s] = v;
                    else if constexpr (DT == DT_F32) out[k * ns + s] = prand_dev::u32_to_f32(v);
                    else out[k * ns + s] = prand_dev::u32_to_f64(v);
                }
            }
        }
    }
    g.store(state, ns, s);
}

template <int GEN> cudaError_t launch(cudaStream_t stream, void *state, void *out, uint64_t ns, uint64_t n, int dtype)
{
    if constexpr (GEN == PRAND_MT19937) {
        const unsigned blocks = (unsigned)ceil_div_u64(ns, 4);
        if (dtype == DT_U32) devapi_mt_kernel<DT_U32><<<blocks, 128, 0, stream>>>(state, (uint32_t *)out, ns, n);
        else if (dtype == DT_F32) devapi_mt_kernel<DT_F32><<<blocks, 128, 0, stream>>>(state, (float *)out, ns, n);
        else devapi_mt_kernel<DT_F64><<<blocks, 128, 0, stream>>>(state, (double *)out, ns, n);
        return cudaGetLastError();
    }
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

cudaError_t devapi_init_generate(cudaStream_t stream, int gen, const void *base, const void *ops, void *out, uint64_t ns,
                                 uint64_t n, int dtype, LaunchInfo *li)
{
    li->kernel = "devapi_init_example";
    li->launches = 1;
    switch (gen) {
    case PRAND_LFSR113: return launch_init<PRAND_LFSR113>(stream, base, ops, out, ns, n, dtype);
    case PRAND_MRG32K3A: return launch_init<PRAND_MRG32K3A>(stream, base, ops, out, ns, n, dtype);
    case PRAND_MT19937: return launch_init<PRAND_MT19937>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GM19: return launch_init<PRAND_GM19>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GM29: return launch_init<PRAND_GM29>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GM31: return launch_init<PRAND_GM31>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GM55: return launch_init<PRAND_GM55>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GM61: return launch_init<PRAND_GM61>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GQ58_1: return launch_init<PRAND_GQ58_1>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GQ58_3: return launch_init<PRAND_GQ58_3>(stream, base, ops, out, ns, n, dtype);
    case PRAND_GQ58_4: return launch_init<PRAND_GQ58_4>(stream, base, ops, out, ns, n, dtype);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace prand
