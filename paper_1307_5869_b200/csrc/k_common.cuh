// k_common.cuh -- device helpers shared by the generation kernels: the fused conversion epilogue
// and the vectorised store path in the canonical layout (a8).
#pragma once
#include <cstdint>
#include "internal.h"

namespace prand {

// ---- conversions ("uniformly distributed in [0,1)"; reading CONV) -----
// f32 = (u >> 8) * 2^-24: a 24-bit integer converts exactly, the power-of-two scale is exact.
__device__ __forceinline__ float u32_to_f32(uint32_t u)
{
    return __uint2float_rn(u >> 8) * 5.9604644775390625e-08f;
}
// f64 = u * 2^-32, built without a conversion instruction: the double with exponent 2^20 and low
// mantissa word u is 2^20 + u * 2^-32 exactly; one exact subtraction removes the offset.
__device__ __forceinline__ double u32_to_f64(uint32_t u)
{
    return __hiloint2double(0x41300000, (int)u) - 1048576.0;
}

template <int DT> struct OutElem;
template <> struct OutElem<DT_U32> { typedef uint32_t type; };
template <> struct OutElem<DT_F32> { typedef float type; };
template <> struct OutElem<DT_F64> { typedef double type; };

template <int DT> __device__ __forceinline__ typename OutElem<DT>::type convert(uint32_t u);
template <> __device__ __forceinline__ uint32_t convert<DT_U32>(uint32_t u) { return u; }
template <> __device__ __forceinline__ float convert<DT_F32>(uint32_t u) { return u32_to_f32(u); }
template <> __device__ __forceinline__ double convert<DT_F64>(uint32_t u) { return u32_to_f64(u); }

// Streaming stores: the output is written once and never re-read by the library, so it should not
// displace anything in L1 (st.global.cs = evict-first).
__device__ __forceinline__ void store1(uint32_t *p, uint32_t a) { __stcs(p, a); }
__device__ __forceinline__ void store1(float *p, float a) { __stcs(p, a); }
__device__ __forceinline__ void store1(double *p, double a) { __stcs(p, a); }

__device__ __forceinline__ void store2(uint32_t *p, uint32_t a, uint32_t b)
{
    __stcs(reinterpret_cast<uint2 *>(p), make_uint2(a, b));
}
__device__ __forceinline__ void store2(float *p, float a, float b)
{
    __stcs(reinterpret_cast<float2 *>(p), make_float2(a, b));
}
__device__ __forceinline__ void store2(double *p, double a, double b)
{
    __stcs(reinterpret_cast<double2 *>(p), make_double2(a, b));
}
__device__ __forceinline__ void store4(uint32_t *p, uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    __stcs(reinterpret_cast<uint4 *>(p), make_uint4(a, b, c, d));
}
__device__ __forceinline__ void store4(float *p, float a, float b, float c, float d)
{
    __stcs(reinterpret_cast<float4 *>(p), make_float4(a, b, c, d));
}
__device__ __forceinline__ void store4(double *p, double a, double b, double c, double d)
{
    __stcs(reinterpret_cast<double2 *>(p), make_double2(a, b));
    __stcs(reinterpret_cast<double2 *>(p) + 1, make_double2(c, d));
}

// Store V consecutive stream values of one row.
template <int V, class T> __device__ __forceinline__ void store_vec(T *p, const T (&v)[V])
{
    if constexpr (V == 1) store1(p, v[0]);
    else if constexpr (V == 2) store2(p, v[0], v[1]);
    else { static_assert(V == 4, "V must be 1, 2 or 4"); store4(p, v[0], v[1], v[2], v[3]); }
}

__host__ __device__ inline uint64_t ceil_div_u64(uint64_t a, uint64_t b) { return (a + b - 1) / b; }

}  // namespace prand
