/* prand_device.cuh -- device-callable single-stream generators.
 *
 * PAPER.md:410, 431-446, 478-511 (sections 7.2-7.4): every PRAND generator can be called from inside a
 * user's CUDA kernel -- `rng_generate_(state)`, `rng_generate_uniform_float_(state)` -- on a state
 * that was initialised by the library or, on the device itself, by `rng_dev_init_sequence_` /
 * `rng_dev_skipahead_` over constant tables placed in device memory (`mrg32k3a_init_device_consts_`).
 * This header is that interface for libprand: header-only `__device__` code, one small struct per
 * generator.
 *
 *   host:    prand_state *st;   prand_init(&st, PRAND_GM31, seed, 1, 0, 0, stream);      // the base stream
 *            const void *base = prand_state_device_ptr(st);
 *            const void *ops;   prand_device_ops(st, L_mant, L_log2, 20, &ops, stream);  // jumps of L * 2^j
 *   device:  prand_dev::Gen<PRAND_GM31> g;
 *            g.load(base, 1, 0);                               // the base stream ...
 *            g.skipahead((const prand_gm_op *)ops, s);         // ... advanced s * L: stream s of the family
 *            uint32_t u = g.next_u32();  float f = g.next_f32();  double x = g.next_f64();
 *            g.store(d_state, n_streams, s);                   // optional: continue later / elsewhere
 *
 * `load / store` also work on the library's own multi-stream state (prand_state_device_ptr of a state
 * with n_streams streams): a stream advanced n times here and exported equals the same stream after
 * prand_generate_*(n).  Semantics are those of include/prand.h: `next_*` returns the stream's next
 * output (step-then-output, reading POS) with the conversions of reading CONV (MRG32K3A
 * f64: reading M3).  `skipahead(ops, idx)` applies ops[b] for every set bit b of idx, i.e. advances the
 * stream by idx * dist when ops came from prand_device_ops(dist, levels > log2 idx).
 *
 * Device state layout (what prand_state_device_ptr returns; owned by the library):
 *   LFSR113, MRG32K3A, GM/GQ: word w of stream s at base[w * n_streams + s], words as in the canonical
 *       export of include/prand.h (u32 words; u64 for GM55, GM61, GQ58.x);
 *   MT19937: stream s's 624-word window x_P..x_{P+623} at base[s * 624 ..].
 *
 * MT19937 is cooperative: `Gen<PRAND_MT19937>` is driven by a whole warp on a 624-word window in
 * shared memory (lane k receives output number 32 c + k of call c), and its skip-ahead
 * (`mt19937_skipahead_cta`, eq. 10 of the paper) by a whole CTA with ~83 KB of dynamic shared memory.
 *
 * The step, output and skip functions below are the ones libprand's own kernels use
 * (paper_1307_5869_b200/csrc/k_*.cu include this header): one definition of the arithmetic.
 * Product code: shares nothing with oracle/.
 */
#pragma once
#include <stdint.h>
#include "prand.h"
#include "prand_ops.h"

namespace prand_dev {

/* ---- conversions (reading CONV): exact ------------------------------ */
__device__ __forceinline__ float u32_to_f32(uint32_t u) { return __uint2float_rn(u >> 8) * 5.9604644775390625e-08f; }
__device__ __forceinline__ double u32_to_f64(uint32_t u) { return __hiloint2double(0x41300000, (int)u) - 1048576.0; }

template <int GEN> struct Gen;

/* ==== LFSR113 (eqs. 7-8 in word form) ==============================================
 * component (p, q, s): z' = ((z & top_p) << s) ^ (((z << q) ^ z) >> (p - s)); output = XOR of the four. */
template <int P, int Q, int S> __device__ __forceinline__ uint32_t tausworthe(uint32_t z)
{
    constexpr uint32_t kept = (0xFFFFFFFFu << (32 - P)) << S;   // (z & top_p) << s == (z << s) & kept
    const uint32_t b = ((z << Q) ^ z) >> (P - S);
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
/* n steps of a component are a GF(2)-linear map of its word, stored by columns (prand_lfsr113_op) */
__device__ __forceinline__ uint32_t gf2_matvec(const uint32_t *__restrict__ col, uint32_t z)
{
    uint32_t r = 0;
#pragma unroll 8
    for (int j = 0; j < 32; j++) r ^= (0u - ((z >> j) & 1u)) & __ldg(col + j);
    return r;
}
__device__ __forceinline__ void lfsr113_apply_bits(const prand_lfsr113_op *__restrict__ ops, uint64_t idx, uint32_t (&z)[4])
{
    for (int lev = 0; idx != 0; lev++, idx >>= 1)
        if (idx & 1)
            for (int c = 0; c < 4; c++) z[c] = gf2_matvec(ops[lev].col[c], z[c]);
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
    __device__ void skipahead(const prand_lfsr113_op *ops, uint64_t idx) { lfsr113_apply_bits(ops, idx, z); }
    __device__ uint32_t next_u32() { return lfsr113_step(z); }
    __device__ float next_f32() { return u32_to_f32(next_u32()); }
    __device__ double next_f64() { return u32_to_f64(next_u32()); }
};

/* ==== MRG32K3A (eqs. 5-6; output reading M1, f64 reading M3) =======================
 *   x_{n+1} = a x_{n-1} + b x_{n-2} mod m1,  a = 1403580, b = -810728,  m1 = 2^32 - 209,
 *   y_{n+1} = c y_n     + d y_{n-2} mod m2,  c = 527612,  d = -1370589, m2 = 2^32 - 22853. */
constexpr uint32_t MRG_M1 = 4294967087u, MRG_M2 = 4294944443u, MRG_C1 = 209u, MRG_C2 = 22853u;

/* x_{n+1} from (x_{n-1}, x_{n-2}).  t = a x1 + b (m1 - x2) < 2^54, t = hi 2^32 + lo; with the quotient
 * estimate hi + 1:  t - (hi+1) m1 = lo + (hi+1) 209 - 2^32.  If the 32-bit addition carries the difference
 * is the wrapped sum (< 2^30 < m1); otherwise the estimate was one too large and adding m1 back gives
 * sum - 209 in [0, m1).  Either way canonical.  c1 = 209 (an opaque register copy in hot loops). */
__device__ __forceinline__ uint32_t mrg_next_x(uint32_t x1, uint32_t x2, uint32_t c1)
{
    uint64_t t = (uint64_t)1403580u * x1 + (uint64_t)810728u * (MRG_M1 - x2);
    uint32_t p = (uint32_t)(t >> 32) * c1 + c1;          // (hi + 1) * 209 < 2^30
    uint32_t s = (uint32_t)t + p;
    return s >= p ? s - MRG_C1 : s;                      // s >= p  <=>  no carry
}
/* y_{n+1} from (y_n, y_{n-2}).  One 64-bit fold u = hi 22853 + lo (< 2^38, same residue; the carry chain
 * keeps it out of a register pair), then the same estimate-and-correct step on u = uh 2^32 + ul. */
__device__ __forceinline__ uint32_t mrg_next_y(uint32_t y0, uint32_t y2)
{
    uint64_t t = (uint64_t)527612u * y0 + (uint64_t)1370589u * (MRG_M2 - y2);
    uint64_t f = (uint64_t)(uint32_t)(t >> 32) * MRG_C2;     // u = f + lo(t), kept as (uh + 1, ul)
    uint32_t ul, uh1;
    asm("add.cc.u32 %0, %2, %3;\n\taddc.u32 %1, %4, 1;"
        : "=r"(ul), "=r"(uh1) : "r"((uint32_t)f), "r"((uint32_t)t), "r"((uint32_t)(f >> 32)));
    uint32_t p = uh1 * MRG_C2;                           // (uh + 1) * 22853 < 2^21
    uint32_t s = ul + p;
    return s >= p ? s - MRG_C2 : s;
}
/* generic a*b mod m for the (cold) skip path: a, b < m = 2^32 - cfold */
__device__ __forceinline__ uint32_t mrg_mulmod(uint32_t a, uint32_t b, uint32_t m, uint32_t cfold)
{
    uint64_t t = (uint64_t)a * b;
    for (int k = 0; k < 3; k++) t = (t >> 32) * cfold + (uint32_t)t;   // < 2^32 + cfold after 3 folds
    while (t >= m) t -= m;
    return (uint32_t)t;
}
__device__ __forceinline__ uint32_t mrg_addmod(uint32_t a, uint32_t b, uint32_t m)
{
    uint64_t t = (uint64_t)a + b;
    return (uint32_t)(t >= m ? t - m : t);
}
__device__ __forceinline__ void mrg_matvec3(const uint32_t *__restrict__ mt, uint32_t &v0, uint32_t &v1, uint32_t &v2,
                                            uint32_t m, uint32_t cfold)
{
    uint32_t r[3];
    for (int i = 0; i < 3; i++) {
        uint32_t acc = mrg_mulmod(__ldg(mt + 3 * i), v0, m, cfold);
        acc = mrg_addmod(acc, mrg_mulmod(__ldg(mt + 3 * i + 1), v1, m, cfold), m);
        acc = mrg_addmod(acc, mrg_mulmod(__ldg(mt + 3 * i + 2), v2, m, cfold), m);
        r[i] = acc;
    }
    v0 = r[0]; v1 = r[1]; v2 = r[2];
}
template <> struct Gen<PRAND_MRG32K3A> {
    static constexpr uint32_t M1 = MRG_M1, M2 = MRG_M2;
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
    __device__ void apply(const prand_mrg32k3a_op *op)
    {
        mrg_matvec3(op->a, x0, x1, x2, MRG_M1, MRG_C1);
        mrg_matvec3(op->b, y0, y1, y2, MRG_M2, MRG_C2);
    }
    __device__ void skipahead(const prand_mrg32k3a_op *ops, uint64_t idx)
    {
        for (int lev = 0; idx != 0; lev++, idx >>= 1)
            if (idx & 1) apply(ops + lev);
    }
    __device__ void step()
    {
        const uint32_t nx = mrg_next_x(x1, x2, MRG_C1), ny = mrg_next_y(y0, y2);
        x2 = x1; x1 = x0; x0 = nx;
        y2 = y1; y1 = y0; y0 = ny;
    }
    __device__ uint32_t next_u32() { step(); return x0 >= y0 ? x0 - y0 : x0 - y0 + M1; }
    __device__ float next_f32() { return u32_to_f32(next_u32()); }
    __device__ double next_f64()
    {
        const uint32_t z = next_u32();
        return (double)(z ? z : M1) * 2.328306549295727688e-10;     /* one IEEE multiply (reading M3) */
    }
};

/* ==== MT19937 (parameters: DESIGN.md reading T1) ====================================
 *   x_{i+624} = x_{i+397} ^ (y >> 1) ^ (y odd ? 0x9908B0DF : 0),  y = (x_i & 0x80000000) | (x_{i+1} & 0x7FFFFFFF),
 *   output number P = temper(x_{P+624}); the state at position P is the window x_P..x_{P+623}. */
constexpr int MT_N = 624, MT_M = 397, MT_DEG = 19937;
__device__ __forceinline__ uint32_t mt_recur(uint32_t xi, uint32_t xi1, uint32_t xim)
{
    uint32_t y = (xi & 0x80000000u) | (xi1 & 0x7FFFFFFFu);
    return xim ^ (y >> 1) ^ ((0u - (y & 1u)) & 0x9908B0DFu);
}
__device__ __forceinline__ uint32_t mt_temper(uint32_t x)
{
    x ^= x >> 11;
    x ^= (x << 7) & 0x9D2C5680u;
    x ^= (x << 15) & 0xEFC60000u;
    x ^= x >> 18;
    return x;
}

/* Warp-cooperative generator.  All 32 lanes of a warp call every member together; `window` points to
 * MT_N words of shared memory owned by the warp for the lifetime of the object.  The window is a circular
 * buffer (cell c holds the latest x_n with n = c mod 624, head = cell of x_P); a call of next_u32
 * regenerates the 32 cells head .. head+31 (any 227 consecutive words are independent) and
 * returns output number P + k to lane k. */
template <> struct Gen<PRAND_MT19937> {
    uint32_t *win;
    int head;
    __device__ void attach(uint32_t *window) { win = window; head = 0; }
    __device__ void load(const void *base, uint64_t, uint64_t s)
    {
        const uint32_t *b = static_cast<const uint32_t *>(base) + s * MT_N;
        for (int j = threadIdx.x & 31; j < MT_N; j += 32) win[j] = b[j];
        head = 0;
        __syncwarp();
    }
    __device__ void store(void *base, uint64_t, uint64_t s) const
    {
        uint32_t *b = static_cast<uint32_t *>(base) + s * MT_N;
        __syncwarp();
        for (int j = threadIdx.x & 31; j < MT_N; j += 32) {
            const int c = head + j;
            b[j] = win[c < MT_N ? c : c - MT_N];
        }
    }
    __device__ uint32_t next_u32()
    {
        const int lane = threadIdx.x & 31;
        int c0 = head + lane, c1 = c0 + 1, cm = c0 + MT_M;
        c0 -= c0 >= MT_N ? MT_N : 0;
        c1 -= c1 >= MT_N ? MT_N : 0;
        cm -= cm >= MT_N ? MT_N : 0;
        cm -= cm >= MT_N ? MT_N : 0;
        const uint32_t x = mt_recur(win[c0], win[c1], win[cm]);
        __syncwarp();                                        /* every operand read before any cell is rewritten */
        win[c0] = x;
        __syncwarp();
        head += 32;
        head -= head >= MT_N ? MT_N : 0;
        return mt_temper(x);
    }
    __device__ float next_f32() { return u32_to_f32(next_u32()); }
    __device__ double next_f64() { return u32_to_f64(next_u32()); }
    /* a single number (all lanes call, every lane receives it): the stream advances by one */
    __device__ uint32_t next_one()
    {
        int c1 = head + 1, cm = head + MT_M;
        c1 -= c1 >= MT_N ? MT_N : 0;
        cm -= cm >= MT_N ? MT_N : 0;
        const uint32_t x = mt_recur(win[head], win[c1], win[cm]);
        __syncwarp();
        if ((threadIdx.x & 31) == 0) win[head] = x;
        __syncwarp();
        head = c1;
        return mt_temper(x);
    }
};

/* CTA-cooperative skip-ahead (eq. 10 in correlation form): window <- g(A) window for the polynomial
 * g = *op.  All NT threads of the CTA call it together; `work` is MT_SKIP_WORK_BYTES of shared memory
 * (16-byte aligned); `src` / `dst` are 624-word windows in global or shared memory (src == dst allowed).
 * The source window is extended to x_0..x_{19937+623} in shared memory (227 independent words per round,
 * PAPER.md:400), then output word j is the XOR of x_{i+j} over the set coefficients a_i.  The
 * coefficients are expanded, 2048 at a time, into a list of set positions, so that the accumulation
 * loop has no bit scan and runs eight positions (24 independent shared loads per thread) at a time; the
 * list is padded with a position whose words are zero.  out0 / NOUT: the range of output words this CTA
 * accumulates (libprand splits one application over several CTAs when few are in flight). */
constexpr int MT_SKIP_XWORDS = MT_DEG + MT_N;                  /* 20561 */
constexpr int MT_SKIP_ZPAD = 771;                              /* zero words after x: >= 768, keeps the list 16-byte aligned */
constexpr int MT_SKIP_CHUNK = 64;                              /* polynomial words per expansion */
constexpr int MT_SKIP_LIST = MT_SKIP_CHUNK * 32 + 8;           /* positions (u16) incl. padding */
constexpr size_t MT_SKIP_WORK_BYTES = (size_t)(MT_SKIP_XWORDS + MT_SKIP_ZPAD) * sizeof(uint32_t) + MT_SKIP_LIST * sizeof(uint16_t) + 16;

template <int NT, int NOUT = MT_N>
__device__ __forceinline__ void mt19937_skipahead_cta(uint32_t *work, const prand_mt19937_op *__restrict__ op,
                                                      const uint32_t *src, uint32_t *dst, const int out0 = 0)
{
    constexpr int nout = NOUT;
    uint32_t *x = work;                                                          /* MT_SKIP_XWORDS + MT_SKIP_ZPAD */
    uint16_t *list = reinterpret_cast<uint16_t *>(work + MT_SKIP_XWORDS + MT_SKIP_ZPAD);   /* MT_SKIP_LIST */
    int *meta = reinterpret_cast<int *>(list + MT_SKIP_LIST);                    /* [0] warp-0 total, [1] count */
    const int tid = threadIdx.x;
    constexpr int NO = (NOUT + NT - 1) / NT;
    __syncthreads();                                                             /* work may still be in use by the caller */
    for (int j = tid; j < MT_N; j += NT) x[j] = src[j];
    for (int j = tid; j < MT_SKIP_ZPAD; j += NT) x[MT_SKIP_XWORDS + j] = 0;
    __syncthreads();
    constexpr int EXT = NT < MT_N - MT_M ? NT : MT_N - MT_M;   /* at most 227 new words are independent */
    for (int r0 = 0; r0 < MT_DEG; r0 += EXT) {
        int k = r0 + tid;
        if (tid < EXT && k < MT_DEG) x[MT_N + k] = mt_recur(x[k], x[k + 1], x[k + MT_M]);
        __syncthreads();
    }
    /* thread t accumulates output words out0 + t, out0 + t + NT, ... (those below out0 + nout) */
    uint32_t acc[NO];
    const uint32_t *xo[NO];
#pragma unroll
    for (int o = 0; o < NO; o++) {
        acc[o] = 0;
        xo[o] = x + (tid + NT * o < nout ? out0 + tid + NT * o : 0);
    }
    for (int c0 = 0; c0 < MT_N; c0 += MT_SKIP_CHUNK) {
        /* expand polynomial words c0 .. c0+63 (threads 0..63, two warps) into the list of set positions */
        if (tid < MT_SKIP_CHUNK) {
            const int wi = c0 + tid;
            uint32_t pw = wi < MT_N ? __ldg(&op->w[wi]) : 0u;
            const int cnt = __popc(pw);
            int incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
                if ((tid & 31) >= d) incl += v;
            }
            if (tid == 31) meta[0] = incl;
            __syncwarp();
            asm volatile("bar.sync 1, 64;" ::: "memory");
            int pos = incl - cnt + (tid >= 32 ? meta[0] : 0);
            if (tid == MT_SKIP_CHUNK - 1) meta[1] = pos + cnt;
            while (pw) {
                list[pos++] = (uint16_t)(wi * 32 + (__ffs(pw) - 1));
                pw &= pw - 1;
            }
        }
        __syncthreads();
        const int n = meta[1];
        if (tid < 8) list[n + tid] = (uint16_t)MT_SKIP_XWORDS;
        __syncthreads();
        for (int k = 0; k < n; k += 8) {
            const uint4 q = *reinterpret_cast<const uint4 *>(list + k);      /* eight positions, uniform */
            const uint32_t ii[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int h = 0; h < 4; h++) {
                const int ia = ii[h] & 0xFFFF, ib = ii[h] >> 16;
#pragma unroll
                for (int o = 0; o < NO; o++) acc[o] ^= xo[o][ia] ^ xo[o][ib];
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int o = 0; o < NO; o++) {
        const int j = out0 + tid + NT * o;
        if (tid + NT * o < nout) dst[j] = j == 0 ? (acc[o] & 0x80000000u) : acc[o];   /* only the top bit of word 0 is state (T2) */
    }
    __syncthreads();
}

}  /* namespace prand_dev */

#include "prand_device_gm.cuh"
