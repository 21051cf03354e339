// k_mrg32k3a.cu -- MRG32K3A jump and generation kernels.
//
// PAPER.md:336-347 (eqs. 5-6): X_{n+1} = A X_n mod m1, Y_{n+1} = B Y_n mod m2 with
//   x_{n+1} = a x_{n-1} + b x_{n-2} mod m1,  a = 1403580, b = -810728,  m1 = 2^32 - 209,
//   y_{n+1} = c y_n     + d y_{n-2} mod m2,  c = 527612,  d = -1370589, m2 = 2^32 - 22853.
// Output (reading M1): z_n = (x_n - y_n) mod m1; f64 = (z_n ? z_n : m1) * 1/(m1+1) (M3).
// Reduction uses 2^32 = 209 (mod m1) and 2^32 = 22853 (mod m2): fold the high word down twice.
// State layout (SoA): word w of stream s at st[w * n_streams + s], w = x_n, x_{n-1}, x_{n-2},
// y_n, y_{n-1}, y_{n-2}.
#include <cstdlib>
#include "k_common.cuh"
#include "../../include/prand_device.cuh"

namespace prand {
namespace {

// recurrences, reduction and the 3x3 skip are the device-callable API's (one definition of the arithmetic)
constexpr uint32_t M1 = prand_dev::MRG_M1, M2 = prand_dev::MRG_M2, C1 = prand_dev::MRG_C1, C2 = prand_dev::MRG_C2;
using prand_dev::mrg_next_x;
using prand_dev::mrg_next_y;
// small CTAs: with ~1000 CTAs on 148 SMs the most loaded SM is within 2% of the average
constexpr int GEN_THREADS = 128;

struct Mrg { uint32_t x0, x1, x2, y0, y1, y2; };   // x0 = x_n, x1 = x_{n-1}, x2 = x_{n-2}

// Output of the combined generator from canonical x < m1, y < m2 < m1 (reading M1):
// z = (x - y) mod m1 in [0, m1); the f64 map sends z = 0 to m1 (reading M3), i.e. z in [1, m1].
template <int DT> __device__ __forceinline__ typename OutElem<DT>::type mrg_output(uint32_t x, uint32_t y)
{
    uint32_t z = x - y;
    if constexpr (DT == DT_F64) {
        if (x <= y) z += M1;
        // one IEEE double multiply of an exactly converted integer
        return (double)z * 2.328306549295727688e-10;
    } else {
        if (x < y) z += M1;
        return convert<DT>(z);
    }
}

__device__ __forceinline__ void matvec3(const uint32_t *__restrict__ mt, uint32_t &v0, uint32_t &v1,
                                        uint32_t &v2, uint32_t m, uint32_t cfold)
{
    prand_dev::mrg_matvec3(mt, v0, v1, v2, m, cfold);
}
__device__ __forceinline__ void mrg_apply_bits(const MrgOp *__restrict__ ops, uint64_t idx, Mrg &s)
{
    for (int lev = 0; idx != 0; lev++, idx >>= 1)
        if (idx & 1) {
            matvec3(ops[lev].a, s.x0, s.x1, s.x2, M1, C1);
            matvec3(ops[lev].b, s.y0, s.y1, s.y2, M2, C2);
        }
}

__device__ __forceinline__ Mrg mrg_load(const uint32_t *st, uint64_t ns, uint64_t s)
{
    Mrg r;
    r.x0 = st[s]; r.x1 = st[ns + s]; r.x2 = st[2 * ns + s];
    r.y0 = st[3 * ns + s]; r.y1 = st[4 * ns + s]; r.y2 = st[5 * ns + s];
    return r;
}
__device__ __forceinline__ void mrg_store(uint32_t *st, uint64_t ns, uint64_t s, const Mrg &r)
{
    st[s] = r.x0; st[ns + s] = r.x1; st[2 * ns + s] = r.x2;
    st[3 * ns + s] = r.y0; st[4 * ns + s] = r.y1; st[5 * ns + s] = r.y2;
}

__global__ void __launch_bounds__(256)
mrg32k3a_jump_kernel(const uint32_t *__restrict__ base, const uint32_t *st_in,
                     uint32_t *st_out, uint64_t ns, const MrgOp *__restrict__ ops,
                     uint64_t idx0, uint64_t idx_stride)
{
    uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    Mrg r;
    if (base) { r.x0 = base[0]; r.x1 = base[1]; r.x2 = base[2]; r.y0 = base[3]; r.y1 = base[4]; r.y2 = base[5]; }
    else r = mrg_load(st_in, ns, s);
    mrg_apply_bits(ops, idx0 + s * idx_stride, r);
    mrg_store(st_out, ns, s, r);
}

__device__ __forceinline__ void mrg_apply_op(const MrgOp *__restrict__ op, Mrg &s)
{
    matvec3(op->a, s.x0, s.x1, s.x2, M1, C1);
    matvec3(op->b, s.y0, s.y1, s.y2, M2, C2);
}

// One thread owns V adjacent streams and one row chunk: blockIdx.y = chunk c, so the row index is
// uniform over the block.  Threads of a warp own adjacent stream groups: a warp writes 32*V
// consecutive elements of a row per step (one 128-bit store per thread for V*sizeof(T) = 16).
// The three-row body renames the state registers instead of moving them:
//   (x_n, x_{n-1}, x_{n-2}) = (a,b,c) -> (c',a,b) -> (b',c',a) -> (a',b',c').
template <int V, int DT>
__global__ void __launch_bounds__(GEN_THREADS)
mrg32k3a_gen_kernel(const uint32_t *st_in, uint32_t *st_out,
                    typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n,
                    uint64_t chunk_len, const MrgOp *__restrict__ chunk_ops)
{
    typedef typename OutElem<DT>::type T;
    const uint64_t sg = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t s0 = sg * V;
    if (s0 >= ns) return;
    const uint32_t c = blockIdx.y;

    Mrg g[V];
#pragma unroll
    for (int v = 0; v < V; v++) g[v] = mrg_load(st_in, ns, s0 + v);
    if (c != 0) {
#pragma unroll
        for (int v = 0; v < V; v++) mrg_apply_op(chunk_ops + (c - 1), g[v]);
    }
    const uint64_t row0 = (uint64_t)c * chunk_len;
    const uint64_t rows = (row0 + chunk_len < n) ? chunk_len : n - row0;
    T *p = out + row0 * ns + s0;
    T r[V];
    // the fold constants as opaque register values: as literals ptxas re-materialises them (one
    // immediate per IMAD) inside the loop
    uint32_t c1 = C1;
    asm volatile("" : "+r"(c1));
    uint64_t i = 0;
#pragma unroll 1
    for (; i + 3 <= rows; i += 3) {
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].x2 = mrg_next_x(g[v].x1, g[v].x2, c1);
            g[v].y2 = mrg_next_y(g[v].y0, g[v].y2);
            r[v] = mrg_output<DT>(g[v].x2, g[v].y2);
        }
        store_vec<V>(p, r);
        p += ns;
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].x1 = mrg_next_x(g[v].x0, g[v].x1, c1);
            g[v].y1 = mrg_next_y(g[v].y2, g[v].y1);
            r[v] = mrg_output<DT>(g[v].x1, g[v].y1);
        }
        store_vec<V>(p, r);
        p += ns;
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].x0 = mrg_next_x(g[v].x2, g[v].x0, c1);
            g[v].y0 = mrg_next_y(g[v].y1, g[v].y0);
            r[v] = mrg_output<DT>(g[v].x0, g[v].y0);
        }
        store_vec<V>(p, r);
        p += ns;
    }
#pragma unroll 1
    for (; i < rows; i++) {                              // ragged tail: rotate by moving
#pragma unroll
        for (int v = 0; v < V; v++) {
            uint32_t nx = mrg_next_x(g[v].x1, g[v].x2, c1), ny = mrg_next_y(g[v].y0, g[v].y2);
            g[v].x2 = g[v].x1; g[v].x1 = g[v].x0; g[v].x0 = nx;
            g[v].y2 = g[v].y1; g[v].y1 = g[v].y0; g[v].y0 = ny;
            r[v] = mrg_output<DT>(nx, ny);
        }
        store_vec<V>(p, r);
        p += ns;
    }
    if (c == gridDim.y - 1) {
#pragma unroll
        for (int v = 0; v < V; v++) mrg_store(st_out, ns, s0 + v, g[v]);
    }
}

// ---- second component on the FP64 pipe (u32 / f32 output) --------------------------------------------
// With 4-byte outputs the integer pipes, not HBM, bound the kernel above (ALU 66 %, FMA 42 %).  The
// B200 has a third arithmetic pipe, FP64 (64 lanes/clk/SM), so the y component runs there, exactly:
// y is kept as a double holding a *signed* representative r in [-m2/2, m2/2] (|r| < 2^31);
//   p = 527612 r_n - 1370589 r_{n-2}            |p| <= 1898201 * m2 / 2 < 2^52: every product and the
//                                               fused sum are integers below 2^53, i.e. exact;
//   k = rint(p / m2) as fma(p, 1/m2, 1.5 * 2^52) - 1.5 * 2^52   (any integer within 1 of p/m2 will do);
//   r' = fma(-k, m2, p) = p - k m2               exact, |r'| <= m2/2 (+ a few units).
// Five FP64 instructions and no compare; the canonical residue for the output is r' + (r' < 0 ? m2 : 0)
// after one exact double -> int32 conversion (XU pipe).
struct MrgY { double y0, y1, y2; };
__device__ __forceinline__ double mrg_y_in(uint32_t y) { return y >= 0x80000000u ? (double)y - 4294944443.0 : (double)y; }
__device__ __forceinline__ uint32_t mrg_y_out(double r)
{
    // exact: r is an integer, |r| < 2^31; r + 1.5 * 2^52 has it (two's complement) in its low mantissa
    // word -- one FP64 add instead of a conversion on the slower XU pipe
    const int32_t v = __double2loint(__dadd_rn(r, 6755399441055744.0));
    return (uint32_t)v + (v < 0 ? M2 : 0u);
}
__device__ __forceinline__ double mrg_next_yd(double y0, double y2)
{
    const double t = __dmul_rn(-1370589.0, y2);
    const double p = __fma_rn(527612.0, y0, t);
    const double km = __fma_rn(p, 2.3283188252407387e-10, 6755399441055744.0);    // 1 / m2, 1.5 * 2^52
    const double k = __dadd_rn(km, -6755399441055744.0);
    return __fma_rn(-k, 4294944443.0, p);
}

// Pipe-balanced forms for the 4-byte kernel, whose binding pipe is the ALU pipe (IADD3, ISETP, SHF, LOP3:
// 64 lanes/clk/SM): additions whose operands allow it are written as multiply-adds with opaque register
// multipliers (IMAD, FMA-heavy pipe); the multipliers are kernel arguments so that ptxas cannot turn them back
// into ALU instructions.
struct MrgK { uint32_t c1, neg1, m2; };
__device__ __forceinline__ uint32_t mrg_next_x_b(uint32_t x1, uint32_t x2, const MrgK &k)
{
    const uint32_t nx2 = x2 * k.neg1 + M1;               // M1 - x2 as one IMAD
    uint64_t t = (uint64_t)1403580u * x1 + (uint64_t)810728u * nx2;
    uint32_t p = (uint32_t)(t >> 32) * k.c1 + k.c1;      // (hi + 1) * 209 < 2^30
    uint32_t s = (uint32_t)t + p;
    return s >= p ? s - C1 : s;                          // s >= p  <=>  no carry
}
__device__ __forceinline__ uint32_t mrg_y_out_b(double r, const MrgK &k)
{
    const uint32_t v = (uint32_t)__double2loint(__dadd_rn(r, 6755399441055744.0));
    uint32_t y;                                          // + m2 for a negative representative: SHF + IMAD
    asm("{.reg .u32 t; shr.u32 t, %1, 31; mad.lo.u32 %0, t, %2, %1;}" : "=r"(y) : "r"(v), "r"(k.m2));
    return y;
}

template <int V, int DT>
__global__ void __launch_bounds__(GEN_THREADS)
mrg32k3a_gen_fp64y_kernel(const uint32_t *st_in, uint32_t *st_out,
                          typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n,
                          uint64_t chunk_len, const MrgOp *__restrict__ chunk_ops, const MrgK k)
{
    typedef typename OutElem<DT>::type T;
    const uint64_t sg = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t s0 = sg * V;
    if (s0 >= ns) return;
    const uint32_t c = blockIdx.y;

    Mrg g[V];
    MrgY h[V];
#pragma unroll
    for (int v = 0; v < V; v++) {
        g[v] = mrg_load(st_in, ns, s0 + v);
        if (c != 0) mrg_apply_op(chunk_ops + (c - 1), g[v]);
        h[v].y0 = mrg_y_in(g[v].y0); h[v].y1 = mrg_y_in(g[v].y1); h[v].y2 = mrg_y_in(g[v].y2);
    }
    const uint64_t row0 = (uint64_t)c * chunk_len;
    const uint64_t rows = (row0 + chunk_len < n) ? chunk_len : n - row0;
    T *p = out + row0 * ns + s0;
    T r[V];
    uint64_t i = 0;
#pragma unroll 1
    for (; i + 3 <= rows; i += 3) {
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].x2 = mrg_next_x_b(g[v].x1, g[v].x2, k);
            h[v].y2 = mrg_next_yd(h[v].y0, h[v].y2);
            r[v] = mrg_output<DT>(g[v].x2, mrg_y_out_b(h[v].y2, k));
        }
        store_vec<V>(p, r);
        p += ns;
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].x1 = mrg_next_x_b(g[v].x0, g[v].x1, k);
            h[v].y1 = mrg_next_yd(h[v].y2, h[v].y1);
            r[v] = mrg_output<DT>(g[v].x1, mrg_y_out_b(h[v].y1, k));
        }
        store_vec<V>(p, r);
        p += ns;
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].x0 = mrg_next_x_b(g[v].x2, g[v].x0, k);
            h[v].y0 = mrg_next_yd(h[v].y1, h[v].y0);
            r[v] = mrg_output<DT>(g[v].x0, mrg_y_out_b(h[v].y0, k));
        }
        store_vec<V>(p, r);
        p += ns;
    }
#pragma unroll 1
    for (; i < rows; i++) {                              // ragged tail: rotate by moving
#pragma unroll
        for (int v = 0; v < V; v++) {
            const uint32_t nx = mrg_next_x_b(g[v].x1, g[v].x2, k);
            const double ny = mrg_next_yd(h[v].y0, h[v].y2);
            g[v].x2 = g[v].x1; g[v].x1 = g[v].x0; g[v].x0 = nx;
            h[v].y2 = h[v].y1; h[v].y1 = h[v].y0; h[v].y0 = ny;
            r[v] = mrg_output<DT>(nx, mrg_y_out_b(ny, k));
        }
        store_vec<V>(p, r);
        p += ns;
    }
    if (c == gridDim.y - 1) {
#pragma unroll
        for (int v = 0; v < V; v++) {
            g[v].y0 = mrg_y_out(h[v].y0); g[v].y1 = mrg_y_out(h[v].y1); g[v].y2 = mrg_y_out(h[v].y2);
            mrg_store(st_out, ns, s0 + v, g[v]);
        }
    }
}

// ---- sections of a single sequence, float64 (prand_generate_seq_f64; the paper's Table 7 task) -------
// The array layout is PRAND's contiguous one, out[c * sec_len + i].  A warp owns 32 V
// consecutive sections, lane k the sections k, k + 32, ...  It collects 16 rows of its sections in a
// shared-memory tile (pitch 18 doubles: 16-byte aligned row pairs, 128-bit shared stores and loads conflict-free) and
// writes them section by section: eight lanes store the 128 contiguous bytes of one section's 16 numbers,
// so a warp store covers four full lines.  V = 1 with up to 2^17 sections fills the GPU with one wave of
// 28 warps per SM; V = 2 serves fewer, longer sections.  The last section's state after its last row is
// the state of the whole sequence after `length` numbers: it goes to st_last, no final jump is needed.
constexpr int SEQ_ROWS = 16, SEQ_PITCH = 18;               // tile[section][row], pitch in doubles (16-byte rows pairs)

template <int V>
__global__ void __launch_bounds__(GEN_THREADS, V == 1 ? 7 : 1)
mrg32k3a_seq_f64_kernel(const uint32_t *st_in, uint32_t *st_last, double *__restrict__ out, uint64_t n_sections,
                        uint64_t sec_len, uint64_t length)
{
    __shared__ __align__(16) double tile_all[GEN_THREADS / 32][32 * V * SEQ_PITCH];
    double *tile = tile_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const uint64_t warp_sec0 = ((uint64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u)) * V;   // first section of the warp
    if (warp_sec0 >= n_sections) return;                   // whole warp
    Mrg g[V];
#pragma unroll
    for (int v = 0; v < V; v++) {
        const uint64_t sec = warp_sec0 + 32 * v + lane;
        g[v] = mrg_load(st_in, n_sections, sec < n_sections ? sec : n_sections - 1);
    }
    uint32_t c1 = C1;
    asm volatile("" : "+r"(c1));
    // rows of the warp's sections: sec_len for all but the last section of the array
    const uint64_t last = n_sections - 1;
    const uint64_t last_rows = length - last * sec_len;
    const bool has_last = warp_sec0 + 32 * V > last;       // this warp owns the last section ...
    const int last_v = has_last ? (int)((last - warp_sec0) >> 5) : 0;   // ... as recurrence last_v of lane (last - warp_sec0) % 32
    const bool owns_last = has_last && lane == (int)((last - warp_sec0) & 31);
    constexpr int LPS = SEQ_ROWS / 2;                      // lanes per section: each stores two doubles
    const int sub = lane / LPS, piece = lane % LPS;
    // Warps whose 32 V sections all exist and are all full-length (every warp but the array's last one) take the
    // lean path: no row or section checks, one running pointer, tile offsets as immediates -- the checks, 64-bit
    // address products and snapshot tests of the general path cost more instructions than the recurrence itself
    // (ncu: 41 instructions per number against 27 in the bulk kernel; issue slots bound this kernel, not HBM).
    if (!has_last && warp_sec0 + 32 * V <= n_sections) {
        double *dst0 = out + (warp_sec0 + sub) * sec_len + 2 * piece;
        const uint64_t kstride = (uint64_t)(32 / LPS) * sec_len;
        const double *tsrc = tile + sub * SEQ_PITCH + 2 * piece;
#pragma unroll 1
        for (uint64_t i0 = 0; i0 < sec_len; i0 += SEQ_ROWS) {
#pragma unroll
            for (int r = 0; r < SEQ_ROWS; r += 2) {        // two rows per 128-bit shared store
#pragma unroll
                for (int v = 0; v < V; v++) {
                    double o[2];
#pragma unroll
                    for (int h = 0; h < 2; h++) {
                        const uint32_t nx = mrg_next_x(g[v].x1, g[v].x2, c1), ny = mrg_next_y(g[v].y0, g[v].y2);
                        g[v].x2 = g[v].x1; g[v].x1 = g[v].x0; g[v].x0 = nx;
                        g[v].y2 = g[v].y1; g[v].y1 = g[v].y0; g[v].y0 = ny;
                        o[h] = mrg_output<DT_F64>(nx, ny);
                    }
                    *reinterpret_cast<double2 *>(tile + (32 * v + lane) * SEQ_PITCH + r) = make_double2(o[0], o[1]);
                }
            }
            __syncwarp();
            double *d = dst0 + i0;
#pragma unroll
            for (int k = 0; k < 32 * V / (32 / LPS); k++) {
                const double2 t = *reinterpret_cast<const double2 *>(tsrc + k * (32 / LPS) * SEQ_PITCH);
                store2(d, t.x, t.y);
                d += kstride;
            }
            __syncwarp();
        }
        return;
    }
#pragma unroll 1
    for (uint64_t i0 = 0; i0 < sec_len; i0 += SEQ_ROWS) {
        const int snap = owns_last && last_rows >= i0 && last_rows < i0 + SEQ_ROWS ? (int)(last_rows - i0) : -1;
#pragma unroll
        for (int r = 0; r < SEQ_ROWS; r++) {
            if (r == snap) mrg_store(st_last, 1, 0, g[last_v]);
#pragma unroll
            for (int v = 0; v < V; v++) {
                const uint32_t nx = mrg_next_x(g[v].x1, g[v].x2, c1), ny = mrg_next_y(g[v].y0, g[v].y2);
                g[v].x2 = g[v].x1; g[v].x1 = g[v].x0; g[v].x0 = nx;
                g[v].y2 = g[v].y1; g[v].y1 = g[v].y0; g[v].y0 = ny;
                tile[(32 * v + lane) * SEQ_PITCH + r] = mrg_output<DT_F64>(nx, ny);
            }
        }
        __syncwarp();
#pragma unroll 4
        for (int k = 0; k < 32 * V / (32 / LPS); k++) {
            const int sl = (32 / LPS) * k + sub;           // section within the warp
            const uint64_t sec = warp_sec0 + sl;
            const uint64_t row = i0 + 2 * piece;
            if (sec < n_sections) {
                const uint64_t rows = sec == last ? last_rows : sec_len;
                const double a = tile[sl * SEQ_PITCH + 2 * piece], b = tile[sl * SEQ_PITCH + 2 * piece + 1];
                double *dst = out + sec * sec_len + row;
                if (row + 1 < rows) store2(dst, a, b);
                else if (row < rows) store1(dst, a);
            }
        }
        __syncwarp();
    }
    if (owns_last && last_rows == sec_len) mrg_store(st_last, 1, 0, g[last_v]);
}

// The same for four-byte outputs (u32, f32): one section per thread, blocks of 32 rows in a per-warp tile
// [section][row] (pitch 33 words: conflict-free both ways), written section by section, eight lanes storing the 128
// contiguous bytes of one section's 32 numbers.  Both components on the integer pipes (the FP64-pipe form of the
// bulk kernel pays off only at the HBM rate, which this layout does not reach).  The caller advances the state of
// the sequence itself (prand_jump by `length`).
template <int DT>
__global__ void __launch_bounds__(GEN_THREADS)
mrg32k3a_seq4_kernel(const uint32_t *st_in, typename OutElem<DT>::type *__restrict__ out, uint64_t n_sections,
                     uint64_t sec_len, uint64_t length)
{
    typedef typename OutElem<DT>::type T;
    static_assert(sizeof(T) == 4, "four-byte outputs");
    constexpr int PITCH = 33, LPS = 8, SPP = 4;            // lanes per section (4 numbers each), sections per pass
    __shared__ T tile_all[GEN_THREADS / 32][32 * PITCH];
    T *tile = tile_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const uint64_t warp_sec0 = (uint64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u);
    if (warp_sec0 >= n_sections) return;                   // whole warp
    Mrg g = mrg_load(st_in, n_sections, warp_sec0 + lane < n_sections ? warp_sec0 + lane : n_sections - 1);
    uint32_t c1 = C1;
    asm volatile("" : "+r"(c1));
    const uint64_t last = n_sections - 1, last_rows = length - last * sec_len;
    const bool whole = warp_sec0 + 32 <= n_sections && (warp_sec0 + 32 <= last || last_rows == sec_len);
    const int sub = lane / LPS, piece = lane % LPS;
    T *dst0 = out + (warp_sec0 + sub) * sec_len + 4 * piece;
    const T *tsrc = tile + sub * PITCH + 4 * piece;
#pragma unroll 1
    for (uint64_t i0 = 0; i0 < sec_len; i0 += 32) {        // (sec_len is a multiple of 32)
#pragma unroll
        for (int r = 0; r < 32; r++) {
            const uint32_t nx = mrg_next_x(g.x1, g.x2, c1), ny = mrg_next_y(g.y0, g.y2);
            g.x2 = g.x1; g.x1 = g.x0; g.x0 = nx;
            g.y2 = g.y1; g.y1 = g.y0; g.y0 = ny;
            tile[lane * PITCH + r] = mrg_output<DT>(nx, ny);
        }
        __syncwarp();
        T *d = dst0 + i0;
#pragma unroll
        for (int k = 0; k < 32 / SPP; k++) {
            T v[4];
#pragma unroll
            for (int e = 0; e < 4; e++) v[e] = tsrc[k * SPP * PITCH + e];
            if (whole) {
                store_vec<4>(d, v);
            } else {
                const uint64_t c = warp_sec0 + SPP * k + sub;
                if (c < n_sections) {
                    const uint64_t rows = c == last ? last_rows : sec_len, row = i0 + 4 * piece;
#pragma unroll
                    for (int e = 0; e < 4; e++)
                        if (row + e < rows) store1(d + e, v[e]);
                }
            }
            d += (uint64_t)SPP * sec_len;
        }
        __syncwarp();
    }
}

template <int V, int DT> cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type T;
    const uint64_t groups = a.n_streams / V;
    dim3 grid((unsigned)ceil_div_u64(groups, GEN_THREADS), (unsigned)a.n_chunks);
    const bool int_only = debug_hooks().mrg_int;                       // test hook: integer y component
    if (DT != DT_F64 && !int_only)
        mrg32k3a_gen_fp64y_kernel<V, DT><<<grid, GEN_THREADS, 0, stream>>>(
            (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (T *)a.out, a.n_streams, a.n, a.chunk_len,
            (const MrgOp *)a.chunk_ops, MrgK{C1, 0xFFFFFFFFu, M2});
    else
        mrg32k3a_gen_kernel<V, DT><<<grid, GEN_THREADS, 0, stream>>>(
            (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (T *)a.out, a.n_streams, a.n, a.chunk_len,
            (const MrgOp *)a.chunk_ops);
    return cudaGetLastError();
}

template <int DT> cudaError_t dispatch_v(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    constexpr int VMAX = (DT == DT_F64) ? 2 : 4;   // one 128-bit store per row
    bool vec = (a.n_streams % VMAX == 0) && ((uintptr_t)a.out % 16 == 0);
    li->launches = 1;
    const bool hooked_int = DT != DT_F64 && debug_hooks().mrg_int;      // named apart so that a test can tell it ran
    if (vec) {
        li->kernel = (DT == DT_F64) ? "mrg32k3a_gen<V=2>" : hooked_int ? "mrg32k3a_gen<V=4,int>" : "mrg32k3a_gen<V=4>";
        return launch_gen<VMAX, DT>(stream, a);
    }
    li->kernel = hooked_int ? "mrg32k3a_gen<V=1,int>" : "mrg32k3a_gen<V=1>";
    return launch_gen<1, DT>(stream, a);
}

}  // namespace

cudaError_t mrg32k3a_jump(cudaStream_t stream, const JumpArgs &a, LaunchInfo *li)
{
    unsigned blocks = (unsigned)ceil_div_u64(a.n_streams, 256);
    mrg32k3a_jump_kernel<<<blocks, 256, 0, stream>>>((const uint32_t *)a.base, (const uint32_t *)a.st_in,
                                                     (uint32_t *)a.st_out, a.n_streams,
                                                     (const MrgOp *)a.ops, a.idx0, a.idx_stride);
    li->kernel = "mrg32k3a_jump";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t mrg32k3a_seq_f64(cudaStream_t stream, const void *st_in, void *st_last, double *out, uint64_t n_sections,
                             uint64_t sec_len, uint64_t length, LaunchInfo *li)
{
    // one section per thread when there are enough of them to fill the GPU, else two (more work in flight per thread)
    if (n_sections >= 32768) {
        const uint64_t threads = ceil_div_u64(n_sections, 32) * 32;
        mrg32k3a_seq_f64_kernel<1><<<(unsigned)ceil_div_u64(threads, GEN_THREADS), GEN_THREADS, 0, stream>>>(
            (const uint32_t *)st_in, (uint32_t *)st_last, out, n_sections, sec_len, length);
    } else {
        const uint64_t threads = ceil_div_u64(n_sections, 64) * 32;
        mrg32k3a_seq_f64_kernel<2><<<(unsigned)ceil_div_u64(threads, GEN_THREADS), GEN_THREADS, 0, stream>>>(
            (const uint32_t *)st_in, (uint32_t *)st_last, out, n_sections, sec_len, length);
    }
    li->kernel = "mrg32k3a_seq_f64";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t mrg32k3a_seq4(cudaStream_t stream, const void *st_in, void *out, int dtype, uint64_t n_sections, uint64_t sec_len,
                          uint64_t length, LaunchInfo *li)
{
    const unsigned blocks = (unsigned)ceil_div_u64(ceil_div_u64(n_sections, 32) * 32, GEN_THREADS);
    if (dtype == DT_U32)
        mrg32k3a_seq4_kernel<DT_U32><<<blocks, GEN_THREADS, 0, stream>>>((const uint32_t *)st_in, (uint32_t *)out, n_sections, sec_len, length);
    else
        mrg32k3a_seq4_kernel<DT_F32><<<blocks, GEN_THREADS, 0, stream>>>((const uint32_t *)st_in, (float *)out, n_sections, sec_len, length);
    li->kernel = "mrg32k3a_seq4";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t mrg32k3a_generate(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    switch (a.dtype) {
    case DT_U32: return dispatch_v<DT_U32>(stream, a, li);
    case DT_F32: return dispatch_v<DT_F32>(stream, a, li);
    default: return dispatch_v<DT_F64>(stream, a, li);
    }
}

}  // namespace prand
