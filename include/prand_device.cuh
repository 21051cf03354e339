/* prand_device.cuh -- device-callable single-stream generators.
 *
 * PAPER.md:410, 437-446, 478 (section 7.3, "#include <gm55.h>" / "_gm55.cu"): every PRAND generator can
 * be called from inside a user's CUDA kernel -- `rng_generate_(state)`, `rng_generate_uniform_float_
 * (state)` -- on a state that was initialised by the library (`rng_init_sequence_`) and copied to
 * the device.  This header is that interface for libprand: header-only `__device__` code, one small
 * struct per generator, operating on the library's device-resident state.
 *
 *   prand_state *st;  prand_init(&st, PRAND_GM31, 1, n_streams, mant, log2, stream);
 *   const void *d = prand_state_device_ptr(st);            // structure-of-arrays state, see below
 *   my_kernel<<<...>>>(d, n_streams, ...);
 *
 *   __global__ void my_kernel(const void *d, uint64_t ns, ...) {
 *       prand_dev::Gen<PRAND_GM31> g;
 *       g.load(d, ns, s);                                   // stream s of the family
 *       uint32_t u = g.next_u32();  float f = g.next_f32();  double x = g.next_f64();
 *       g.store(d_mut, ns, s);                              // optional: continue later / elsewhere
 *   }
 *
 * Semantics are those of include/prand.h: `next_*` returns the stream's next output (step-then-
 * output, reading POS) with the conversions of reading CONV (MRG32K3A f64: reading M3); a
 * stream advanced n times here and exported equals the same stream after prand_generate_*(n).
 *
 * Device state layout (what prand_state_device_ptr returns; owned by the library):
 *   LFSR113, MRG32K3A, GM/GQ: word w of stream s at base[w * n_streams + s], words as in the canonical
 *       export of include/prand.h (u32 words; u64 for GM55, GM61, GQ58.x);
 *   MT19937: stream s's 624-word window x_P..x_{P+623} at base[s * 624 ..].
 *
 * The step functions of the GM/GQ family are the ones the bulk kernels of libprand use
 * (paper_1307_5869_b200/csrc/k_gmgq.cu includes this header).  Jump-ahead inside a kernel is not
 * offered here: use prand_jump / prand_init's block splitting, which run the jump kernels.
 * Product code: shares nothing with oracle/.
 */
#pragma once
#include <stdint.h>
#include "prand.h"

namespace prand_dev {

/* ---- conversions (reading CONV): exact ------------------------------ */
__device__ __forceinline__ float u32_to_f32(uint32_t u) { return __uint2float_rn(u >> 8) * 5.9604644775390625e-08f; }
__device__ __forceinline__ double u32_to_f64(uint32_t u) { return __hiloint2double(0x41300000, (int)u) - 1048576.0; }

template <int GEN> struct Gen;

/* ---- LFSR113 (eqs. 7-8 in word form) ---------------------------------------------
 * component (p, q, s): z' = ((z & top_p) << s) ^ (((z << q) ^ z) >> (p - s)); output = XOR of the four. */
template <int P, int Q, int S> __device__ __forceinline__ uint32_t tausworthe_step(uint32_t z)
{
    const uint32_t b = ((z << Q) ^ z) >> (P - S);
    return ((z & (0xFFFFFFFFu << (32 - P))) << S) ^ b;
}
template <> struct Gen<PRAND_LFSR113> {
    uint32_t z[4];
    __device__ void load(const void *base, uint64_t ns, uint64_t s)
    {
        const uint32_t *b = static_cast<const uint32_t *>(base);
        for (int c = 0; c < 4; c++) z[c] = b[c * ns + s];
    }
    __device__ void store(void *base, uint64_t ns, uint64_t s) const
    {
        uint32_t *b = static_cast<uint32_t *>(base);
        for (int c = 0; c < 4; c++) b[c * ns + s] = z[c];
    }
    __device__ uint32_t next_u32()
    {
        z[0] = tausworthe_step<31, 6, 18>(z[0]);
        z[1] = tausworthe_step<29, 2, 2>(z[1]);
        z[2] = tausworthe_step<28, 13, 7>(z[2]);
        z[3] = tausworthe_step<25, 3, 13>(z[3]);
        return z[0] ^ z[1] ^ z[2] ^ z[3];
    }
    __device__ float next_f32() { return u32_to_f32(next_u32()); }
    __device__ double next_f64() { return u32_to_f64(next_u32()); }
};

/* ---- MRG32K3A (eqs. 5-6; output reading M1, f64 reading M3) ------------------------ */
template <> struct Gen<PRAND_MRG32K3A> {
    static constexpr uint32_t M1 = 4294967087u, M2 = 4294944443u;
    uint32_t x0, x1, x2, y0, y1, y2;                         /* x0 = x_n, x1 = x_{n-1}, x2 = x_{n-2} */
    __device__ void load(const void *base, uint64_t ns, uint64_t s)
    {
        const uint32_t *b = static_cast<const uint32_t *>(base);
        x0 = b[s]; x1 = b[ns + s]; x2 = b[2 * ns + s];
        y0 = b[3 * ns + s]; y1 = b[4 * ns + s]; y2 = b[5 * ns + s];
    }
    __device__ void store(void *base, uint64_t ns, uint64_t s) const
    {
        uint32_t *b = static_cast<uint32_t *>(base);
        b[s] = x0; b[ns + s] = x1; b[2 * ns + s] = x2;
        b[3 * ns + s] = y0; b[4 * ns + s] = y1; b[5 * ns + s] = y2;
    }
    __device__ void step()
    {
        /* x_{n+1} = 1403580 x_{n-1} - 810728 x_{n-2} mod m1;  y_{n+1} = 527612 y_n - 1370589 y_{n-2} mod m2 */
        const uint64_t tx = (uint64_t)1403580u * x1 + (uint64_t)810728u * (M1 - x2);
        const uint64_t ty = (uint64_t)527612u * y0 + (uint64_t)1370589u * (M2 - y2);
        x2 = x1; x1 = x0; x0 = (uint32_t)(tx % M1);
        y2 = y1; y1 = y0; y0 = (uint32_t)(ty % M2);
    }
    __device__ uint32_t next_u32() { step(); return x0 >= y0 ? x0 - y0 : x0 - y0 + M1; }
    __device__ float next_f32() { return u32_to_f32(next_u32()); }
    __device__ double next_f64()
    {
        const uint32_t z = next_u32();
        return (double)(z ? z : M1) * 2.328306549295727688e-10;     /* one IEEE multiply (reading M3) */
    }
};

/* ---- MT19937 (parameters: DESIGN.md reading T1) ------------------------------------------
 * The 624-word window lives in the thread's local memory as a circular buffer. */
template <> struct Gen<PRAND_MT19937> {
    uint32_t w[624];
    int h;                                                   /* slot of x_P */
    __device__ void load(const void *base, uint64_t, uint64_t s)
    {
        const uint32_t *b = static_cast<const uint32_t *>(base) + s * 624;
        for (int j = 0; j < 624; j++) w[j] = b[j];
        h = 0;
    }
    __device__ void store(void *base, uint64_t, uint64_t s) const
    {
        uint32_t *b = static_cast<uint32_t *>(base) + s * 624;
        for (int j = 0; j < 624; j++) b[j] = w[(h + j) % 624];
    }
    __device__ uint32_t next_u32()
    {
        const int i1 = h + 1 < 624 ? h + 1 : 0, im = h + 397 < 624 ? h + 397 : h + 397 - 624;
        const uint32_t y = (w[h] & 0x80000000u) | (w[i1] & 0x7FFFFFFFu);
        uint32_t x = w[im] ^ (y >> 1) ^ ((y & 1u) ? 0x9908B0DFu : 0u);
        w[h] = x;
        h = i1;
        x ^= x >> 11;
        x ^= (x << 7) & 0x9D2C5680u;
        x ^= (x << 15) & 0xEFC60000u;
        x ^= x >> 18;
        return x;
    }
    __device__ float next_f32() { return u32_to_f32(next_u32()); }
    __device__ double next_f64() { return u32_to_f64(next_u32()); }
};

}  /* namespace prand_dev */

#include "prand_device_gm.cuh"
