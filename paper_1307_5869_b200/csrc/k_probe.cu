// k_probe.cu -- measurement probes of libprand: the empty-kernel launch floor and the
// per-pipe instruction rates of the B200 SM that DESIGN.md section 6 uses as the integer roofline.
// None of them is on the hot path; bench.py calls them next to the generators so that floors and
// peaks come from the same run.
//
// Pipe-rate probe: every thread runs ILP independent dependency chains of one instruction (inline
// PTX, so that the SASS opcode is the intended one -- checked with `cuobjdump -sass`, see
// profiles/pipe_rates.md) for `iters` iterations; the grid is 8 CTAs x 256 threads per SM, i.e. the
// scheduler always has an eligible warp.  thread-ops / (time x SM clock x SMs) = ops per clock per SM.
#include "k_common.cuh"

namespace prand {
namespace {

__global__ void empty_kernel() {}

enum {
    OP_IMAD = 0, OP_IMAD_WIDE, OP_IMAD_HI, OP_LOP3, OP_SHF, OP_IADD3, OP_VIADDMNMX, OP_PRMT, OP_ISETP_SEL,
    OP_DFMA, OP_DADD, OP_DMUL, OP_I2F_F64, OP_F2I_F64, OP_SHFL, OP_POPC, OP_IMAD_LOP3, OP_IMAD_LOP3_DFMA,
    OP_FFMA, OP_COUNT
};

const char *const OP_NAME[OP_COUNT] = {
    "IMAD (mad.lo.u32)", "IMAD.WIDE.U32 (mad.wide.u32)", "IMAD.HI.U32 (mul.hi.u32)", "LOP3 (lop3.b32)",
    "SHF (shf.l.wrap.b32)", "IADD3 (a + b + c)", "VIADDMNMX (min(a, a - c))", "PRMT (prmt.b32)",
    "ISETP + SEL (setp.lt + selp)", "DFMA (fma.rn.f64)", "DADD (add.rn.f64)", "DMUL (mul.rn.f64)",
    "I2F.F64.U32 (cvt.rn.f64.u32)", "F2I.U32.F64 (cvt.rzi.u32.f64)", "SHFL.BFLY (shfl.sync.bfly)", "POPC (popc.b32)",
    "IMAD + LOP3 alternating", "IMAD + LOP3 + DFMA alternating", "FFMA (fma.rn.f32)"};

constexpr int ILP = 8, UNROLL = 16;

template <int OP> __device__ __forceinline__ void one(uint32_t &a, uint64_t &w, double &d, float &f, uint32_t b, uint32_t c)
{
    if constexpr (OP == OP_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a) : "r"(b), "r"(c));
    else if constexpr (OP == OP_IMAD_WIDE) asm volatile("{.reg .u32 lo; mov.b64 {lo, _}, %0; mad.wide.u32 %0, lo, %1, %0;}" : "+l"(w) : "r"(c));
    else if constexpr (OP == OP_IMAD_HI) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a) : "r"(b));
    else if constexpr (OP == OP_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(c));
    else if constexpr (OP == OP_SHF) asm volatile("shf.l.wrap.b32 %0, %0, %1, %2;" : "+r"(a) : "r"(b), "r"(c));
    else if constexpr (OP == OP_IADD3) asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a) : "r"(b), "r"(c));
    else if constexpr (OP == OP_VIADDMNMX) asm volatile("{.reg .u32 t; sub.u32 t, %0, %1; min.u32 %0, %0, t;}" : "+r"(a) : "r"(c));
    else if constexpr (OP == OP_PRMT) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(a) : "r"(b), "r"(c));
    else if constexpr (OP == OP_ISETP_SEL) asm volatile("{.reg .pred p; setp.lt.u32 p, %0, %1; selp.u32 %0, %2, %0, p;}" : "+r"(a) : "r"(b), "r"(c));
    else if constexpr (OP == OP_DFMA) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d) : "d"(1.0000001), "d"(1e-9));
    else if constexpr (OP == OP_DADD) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d) : "d"(1e-9));
    else if constexpr (OP == OP_DMUL) asm volatile("mul.rn.f64 %0, %0, %1;" : "+d"(d) : "d"(1.0000001));
    else if constexpr (OP == OP_I2F_F64) asm volatile("{.reg .f64 t; cvt.rn.f64.u32 t, %0; mov.b64 {%0, _}, t;}" : "+r"(a));
    else if constexpr (OP == OP_F2I_F64) asm volatile("{.reg .u32 t; cvt.rzi.u32.f64 t, %0; mov.b64 %0, {t, %1};}" : "+d"(d) : "r"(0x41300000u));
    else if constexpr (OP == OP_SHFL) asm volatile("shfl.sync.bfly.b32 %0, %0, %1, 0x1f, 0xffffffff;" : "+r"(a) : "r"(b & 31u));
    else if constexpr (OP == OP_POPC) asm volatile("{.reg .u32 t; popc.b32 t, %0; add.u32 %0, %0, t;}" : "+r"(a));
    else if constexpr (OP == OP_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(1.0000001f), "f"(1e-9f));
}

// thread-ops counted per call of one<OP>: the probes that need a helper instruction to close the chain
// (POPC + add, ISETP + SEL, add x2) count the pair as the unit named in OP_NAME.
template <int OP>
__global__ void __launch_bounds__(256)
pipe_kernel(uint32_t *sink, uint64_t iters, uint32_t b, uint32_t c)
{
    uint32_t a[ILP];
    uint64_t w[ILP];
    double d[ILP];
    float f[ILP];
#pragma unroll
    for (int k = 0; k < ILP; k++) {
        a[k] = threadIdx.x * 2654435761u + k;
        w[k] = a[k];
        d[k] = 1.0 + k;
        f[k] = 1.0f + k;
    }
#pragma unroll 1
    for (uint64_t i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < UNROLL; u++) {
#pragma unroll
            for (int k = 0; k < ILP; k++) {
                if constexpr (OP == OP_IMAD_LOP3) {
                    if (k & 1) one<OP_IMAD>(a[k], w[k], d[k], f[k], b, c);
                    else one<OP_LOP3>(a[k], w[k], d[k], f[k], b, c);
                } else if constexpr (OP == OP_IMAD_LOP3_DFMA) {
                    if (k % 3 == 0) one<OP_IMAD>(a[k], w[k], d[k], f[k], b, c);
                    else if (k % 3 == 1) one<OP_LOP3>(a[k], w[k], d[k], f[k], b, c);
                    else one<OP_DFMA>(a[k], w[k], d[k], f[k], b, c);
                } else {
                    one<OP>(a[k], w[k], d[k], f[k], b, c);
                }
            }
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int k = 0; k < ILP; k++) r ^= a[k] ^ (uint32_t)w[k] ^ (uint32_t)(w[k] >> 32) ^ (uint32_t)__double2loint(d[k]) ^ __float_as_uint(f[k]);
    if (r == 0x12345u && sink) sink[0] = r;                 // keeps the chains alive
}

template <int OP> cudaError_t launch_pipe(cudaStream_t stream, unsigned blocks, uint64_t iters)
{
    pipe_kernel<OP><<<blocks, 256, 0, stream>>>(nullptr, iters, 0x9E3779B9u, 0x7F4A7C15u);
    return cudaGetLastError();
}

}  // namespace
}  // namespace prand

using namespace prand;

extern "C" int prand_probe_empty(void *cuda_stream)
{
    empty_kernel<<<1, 32, 0, (cudaStream_t)cuda_stream>>>();
    return cudaGetLastError() == cudaSuccess ? PRAND_OK : PRAND_ERR_CUDA;
}

extern "C" int prand_probe_memset(void *d_ptr, int value, size_t bytes, void *cuda_stream)
{
    if (!d_ptr && bytes) return PRAND_ERR_ARG;
    return cudaMemsetAsync(d_ptr, value, bytes, (cudaStream_t)cuda_stream) == cudaSuccess ? PRAND_OK : PRAND_ERR_CUDA;
}

extern "C" int prand_probe_pipe_count(void) { return OP_COUNT; }

extern "C" const char *prand_probe_pipe_name(int op) { return (op < 0 || op >= OP_COUNT) ? "" : OP_NAME[op]; }

extern "C" int prand_probe_pipe(int op, uint64_t iters, uint64_t *thread_ops, void *cuda_stream)
{
    if (op < 0 || op >= OP_COUNT || !thread_ops) return PRAND_ERR_ARG;
    const unsigned blocks = (unsigned)sm_count() * 8;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    *thread_ops = (uint64_t)blocks * 256 * ILP * UNROLL * iters;
    cudaError_t e;
    switch (op) {
#define PRAND_PIPE_CASE(X) case X: e = launch_pipe<X>(s, blocks, iters); break;
    PRAND_PIPE_CASE(OP_IMAD) PRAND_PIPE_CASE(OP_IMAD_WIDE) PRAND_PIPE_CASE(OP_IMAD_HI) PRAND_PIPE_CASE(OP_LOP3)
    PRAND_PIPE_CASE(OP_SHF) PRAND_PIPE_CASE(OP_IADD3) PRAND_PIPE_CASE(OP_VIADDMNMX) PRAND_PIPE_CASE(OP_PRMT)
    PRAND_PIPE_CASE(OP_ISETP_SEL) PRAND_PIPE_CASE(OP_DFMA) PRAND_PIPE_CASE(OP_DADD) PRAND_PIPE_CASE(OP_DMUL)
    PRAND_PIPE_CASE(OP_I2F_F64) PRAND_PIPE_CASE(OP_F2I_F64) PRAND_PIPE_CASE(OP_SHFL) PRAND_PIPE_CASE(OP_POPC)
    PRAND_PIPE_CASE(OP_IMAD_LOP3) PRAND_PIPE_CASE(OP_IMAD_LOP3_DFMA) PRAND_PIPE_CASE(OP_FFMA)
#undef PRAND_PIPE_CASE
    default: return PRAND_ERR_ARG;
    }
    return e == cudaSuccess ? PRAND_OK : PRAND_ERR_CUDA;
}
