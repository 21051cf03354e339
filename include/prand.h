/*
 * prand.h -- C ABI of the B200-native PRAND hot path (arXiv 1307.5869, Barash & Shchur).
 *
 * What the library does: it holds `n_streams` independent streams of one
 * generator, initialised by block splitting -- stream s starts at position s*block_len of the single
 * base sequence defined by the seed -- and fills a caller-owned DEVICE array with uniform numbers in
 * the canonical interleaved layout
 *
 *        out[i * n_streams + s]  =  output number i (counted from the stream's current position)
 *                                   of stream s,           0 <= i < n_per_stream, 0 <= s < n_streams.
 *
 * Every step (skip-operator application, the recurrences, conversion, stores) runs in hand-written
 * CUDA kernels for sm_100a; there is no CPU fallback.  The host side only prepares the skip operators
 * and launches.
 *
 * Conventions
 *  - All functions return 0 (PRAND_OK) or a negative prand_error code; prand_strerror() names it.
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Kernel
 *    launches are asynchronous on it.  prand_init / prand_jump may synchronise it while uploading
 *    operator tables; prand_get_state / prand_set_state / *_host synchronise.
 *  - Pointers named `out` / `d_*` are DEVICE pointers, pointers named `host_*` are HOST pointers.
 *  - The state object is opaque, lives on the device that was current in prand_init, and is owned by
 *    the library until prand_free.  One state must not be used from two CUDA streams concurrently.
 *  - Large distances are passed as mant * 2^log2 (the paper itself passes a*2^b to
 *    mt19937_skipahead_, and split words to mrg32k3a_skipahead_).
 *  - Position convention ("step-then-output"): a state at position P yields output number P by
 *    advancing one step and reading the new state.
 */
#ifndef PRAND_H
#define PRAND_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct prand_state prand_state;

/* Generators (Table 2).  Numeric values are part of the ABI. */
enum prand_gen {
    PRAND_LFSR113 = 0,
    PRAND_MRG32K3A = 1,
    PRAND_MT19937 = 2,
    PRAND_GM19 = 3,      /* PAPER.md:281-284, Table 2 */
    PRAND_GM29 = 4,
    PRAND_GM31 = 5,
    PRAND_GM55 = 6,
    PRAND_GM61 = 7,
    PRAND_GQ58_1 = 8,
    PRAND_GQ58_3 = 9,
    PRAND_GQ58_4 = 10,
    PRAND_NGEN = 11
};

enum prand_error {
    PRAND_OK = 0,
    PRAND_ERR_GEN = -1,        /* unknown generator id                                        */
    PRAND_ERR_ARG = -2,        /* null pointer, n_streams == 0, mant == 0 with log2 != 0, ... */
    PRAND_ERR_SEED = -3,       /* seed not valid for the generator (see prand_init)           */
    PRAND_ERR_OVERFLOW = -4,   /* (first_stream + n_streams - 1) * mant does not fit 64 bits  */
    PRAND_ERR_CUDA = -5,       /* a CUDA runtime call failed; prand_last_cuda_error() has it  */
    PRAND_ERR_SIZE = -6,       /* byte count does not match prand_state_bytes()               */
    PRAND_ERR_ALLOC = -7,      /* host or device allocation failed                            */
    PRAND_ERR_INTERNAL = -8,   /* MT19937: the characteristic polynomial failed its self-check  */
    PRAND_ERR_CAPACITY = -9    /* request larger than the fixed capacity of a no-allocation entry point */
};

/*
 * prand_init -- block-splitting stream initialisation (rng_init_sequence_).
 *   Creates `n_streams` streams of generator `gen`; stream s is the base sequence of `seed` advanced
 *   s * block_len steps, block_len = block_len_mant * 2^block_len_log2 (block_len = 0 is allowed:
 *   all streams identical).  Host: builds the skip operators for block_len * 2^j; device: one init
 *   kernel applies them per stream and writes the structure-of-arrays state.
 *   Seed convention: LFSR113 all four words = seed (invalid if any component's significant top bits
 *   are zero, i.e. seed < 128); MRG32K3A all six words = seed (0 < seed < 2^32 - 22853); MT19937 the
 *   ref.-[2] initialiser x_0 = seed, x_i = 1812433253 (x_{i-1} ^ (x_{i-1} >> 30)) + i; GM/GQ: base
 *   orbit w(0) = 0, w(1) = seed mod g (must be non-zero), ensemble point i at orbit offset
 *   (i+1) * 2^d (reading G3).  LFSR113/MRG32K3A/MT19937 seeds must be < 2^32.
 *   `*st` receives the new state; on error it is set to NULL.
 */
int prand_init(prand_state **st, int gen, uint64_t seed, uint64_t n_streams,
               uint64_t block_len_mant, unsigned block_len_log2, void *cuda_stream);

/*
 * prand_init_shard -- as prand_init, but this state holds only global streams
 *   [first_stream, first_stream + n_streams) of the block-split family (multi-GPU sharding by stream
 *   index; streams are independent, so no exchange is needed).  Local stream j is
 *   global stream first_stream + j; the output layout is out[i * n_streams + j].
 */
int prand_init_shard(prand_state **st, int gen, uint64_t seed, uint64_t first_stream,
                     uint64_t n_streams, uint64_t block_len_mant, unsigned block_len_log2,
                     void *cuda_stream);

/*
 * prand_jump -- advance EVERY stream by steps = steps_mant * 2^steps_log2 without generating
 *   (rng_skipahead_; PAPER.md:286-301, 347, 363-370, 374-378 for the algebra).
 */
int prand_jump(prand_state *st, uint64_t steps_mant, unsigned steps_log2, void *cuda_stream);

/*
 * prand_generate_{u32,f32,f64} -- bulk generation (
 *   rng_generate_gpu_array_{,float_,double_}).  `out` is device memory with n_per_stream * n_streams
 *   elements, element-aligned; every stream advances n_per_stream.  Successive calls continue the
 *   streams.  n_per_stream == 0 is a no-op.  There is no divisibility requirement (PAPER.md:404 had
 *   one).  Internally a stream's range may be cut into sub-sections reached by jump-ahead
 *   (PAPER.md:382); this never changes any output.
 *     u32: the generator's 32-bit output word (MRG32K3A: z_n in [0, 2^32-209)).
 *     f32: (u >> 8) * 2^-24 in [0,1)   (reading CONV).
 *     f64: u * 2^-32 in [0,1); MRG32K3A: (z_n ? z_n : m1) / (m1 + 1) in (0,1) (reading M3).
 */
int prand_generate_u32(prand_state *st, uint32_t *out, uint64_t n_per_stream, void *cuda_stream);
int prand_generate_f32(prand_state *st, float *out, uint64_t n_per_stream, void *cuda_stream);
int prand_generate_f64(prand_state *st, double *out, uint64_t n_per_stream, void *cuda_stream);

/*
 * prand_generate_{u32,f32,f64}_host -- the same numbers delivered to HOST memory
 *   (rng_generate_array_): generated on the device in row blocks and copied back with
 *   overlapping device-to-host copies.  `host_out` has n_per_stream * n_streams elements (pinned
 *   memory gives full PCIe speed; pageable memory works).  Returns after the data has arrived.
 */
int prand_generate_u32_host(prand_state *st, uint32_t *host_out, uint64_t n_per_stream, void *cuda_stream);
int prand_generate_f32_host(prand_state *st, float *host_out, uint64_t n_per_stream, void *cuda_stream);
int prand_generate_f64_host(prand_state *st, double *host_out, uint64_t n_per_stream, void *cuda_stream);

/*
 * prand_generate_seq_{u32,f32,f64} -- PRAND's single-sequence array fill ("the output
 *   array is divided into sections ... jumping ahead to a starting point of the section", Table 5
 *   PAPER.md:384-404, rng_generate_gpu_array_ PAPER.md:465).  `st` must hold exactly one stream
 *   (n_streams == 1, else PRAND_ERR_ARG).  out[j], j < length, = output number j of that stream counted
 *   from its current position, i.e. exactly what `length` successive single-stream generate calls
 *   would have produced; afterwards the stream has advanced by `length`.  `out` is caller-owned DEVICE
 *   memory with `length` elements.  Unlike PRAND no divisibility of `length` by the
 *   number of sections is required (MT19937: no power of two).  LFSR113, MRG32K3A and MT19937 write `out`
 *   in place when it is 16-byte aligned; the GM/GQ generators (and unaligned `out`) go through a stream-ordered
 *   scratch buffer of about `length` elements that the library allocates for the duration of the call.
 */
int prand_generate_seq_u32(prand_state *st, uint32_t *out, uint64_t length, void *cuda_stream);
int prand_generate_seq_f32(prand_state *st, float *out, uint64_t length, void *cuda_stream);
int prand_generate_seq_f64(prand_state *st, double *out, uint64_t length, void *cuda_stream);

/*
 * prand_lfsr113_seq_noalloc_u32 -- the single-sequence fill (Table 5) for callers
 *   that must not allocate device memory.
 *
 *   Why it exists: all other generating calls work on a prand_state, which prand_init creates from the library's
 *   memory pool, and prand_generate_seq_* allocates its table of section start states on demand.  Code that runs
 *   where the CUDA allocator is off limits -- inside a latency-critical loop that owns one arena reserved at
 *   start-up, under a framework whose caching allocator owns the device and tolerates no foreign cudaMalloc or
 *   pool growth, in a plug-in that may only use the buffers its host application hands it, or so close to the
 *   memory limit that an allocation could fail or stall the device -- cannot use those calls at that point.  This
 *   one calls no cudaMalloc / cudaFree / pool routine and no library routine that allocates device memory: the
 *   section table and the jump operators live in a fixed 520 KiB __device__ array inside libprand.so (each GPU
 *   that loads the library holds its copy until the process exits).
 *
 *   d_state  DEVICE pointer to 4 x u32, caller-owned: the LFSR113 state in the canonical layout of prand_get_state
 *            for one stream (z1..z4).  Read as the start of the sequence and overwritten with the state after
 *            `length` numbers, so successive calls continue the sequence and the words can be given to
 *            prand_set_state.  The words are not validated here (a component whose significant top bits are all
 *            zero stays zero, as prand_init / prand_set_state would have refused).
 *   out      DEVICE pointer, `length` u32, 16-byte aligned, caller-owned.  out[j] = output number j of the
 *            sequence counted from the state's position: exactly what prand_generate_seq_u32 writes.
 *   length   at most PRAND_NOALLOC_MAX_LENGTH numbers per call (the array holds PRAND_NOALLOC_MAX_SECTIONS
 *            section start states and a section is kept to at most 65,536 numbers); more returns
 *            PRAND_ERR_CAPACITY and nothing is launched -- fill a longer array with several calls.  0 is a no-op.
 *   Errors   PRAND_ERR_ARG (null or misaligned pointer), PRAND_ERR_CAPACITY, PRAND_ERR_CUDA.
 *
 *   The work (two operator uploads of at most 8 KiB from host memory, three kernel launches) is asynchronous on
 *   `cuda_stream`.  The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, with
 *   that device current), which may load the library's module there: make that first call before any stream
 *   capture begins.  All calls on a device share the one array, which keeps what the previous call wrote; nothing
 *   in it needs clearing (each call writes every word it reads), but two calls whose GPU work overlaps -- streams
 *   without an ordering between them, or concurrent host threads -- race on it and give wrong numbers.  Keep the
 *   calls on one stream or order them with events.
 */
#define PRAND_NOALLOC_MAX_SECTIONS 32768u
#define PRAND_NOALLOC_MAX_LENGTH (1ull << 31)
int prand_lfsr113_seq_noalloc_u32(uint32_t *d_state, uint32_t *out, uint64_t length, void *cuda_stream);

/*
 * prand_generate_strided_{u32,f32,f64} -- the generator that skips ahead after every output
 *   (PAPER.md:226 and Table 3: sequences that jump 2^n per step).  out[i * n_streams
 *   + s] = the output of stream s at position P_s + i * stride (P_s = its current position), stride =
 *   stride_mant * 2^stride_log2 >= 1; afterwards every stream has advanced n_per_stream * stride.
 *   One jump per output row (the operator is prepared once): meant for testing skip-ahead sequences,
 *   not for bulk throughput.  The library keeps a second state buffer while it runs (the stepped state of the
 *   output row lands there; the state itself is not copied).
 */
int prand_generate_strided_u32(prand_state *st, uint32_t *out, uint64_t n_per_stream, uint64_t stride_mant,
                               unsigned stride_log2, void *cuda_stream);
int prand_generate_strided_f32(prand_state *st, float *out, uint64_t n_per_stream, uint64_t stride_mant,
                               unsigned stride_log2, void *cuda_stream);
int prand_generate_strided_f64(prand_state *st, double *out, uint64_t n_per_stream, uint64_t stride_mant,
                               unsigned stride_log2, void *cuda_stream);

/*
 * Device-callable API (the generators can be called from a user's kernel).
 * include/prand_device.cuh holds the header-only __device__ generators; these calls give a kernel
 * access to the library's device-resident state (layout documented in that header; the pointer stays
 * valid until the next prand_generate_* call that uses sub-sections, prand_set_state or prand_free)
 * and run the library's own example kernel written against that header: one thread per stream (MT19937:
 * one warp per stream on a shared-memory window),
 * out[i * n_streams + s] as for prand_generate_*, the streams advance by n_per_stream.  The example
 * is a self-test of the header, not a fast path.
 */
/*
 * prand_device_ops -- operator table for skip-ahead INSIDE a user's kernel (PRAND's
 *   `*_init_device_consts_` places the tables that `*_dev_skipahead_` / `*_dev_init_sequence_` use in
 *   device memory).  Builds the skip operators of generator prand_gen_of(st) for the distances
 *   dist * 2^j, j = 0 .. levels-1 (dist = dist_mant * 2^dist_log2), uploads them and returns in *d_ops a
 *   DEVICE pointer to an array of `levels` operators (prand_lfsr113_op / prand_mrg32k3a_op /
 *   prand_mt19937_op / prand_gm_op of include/prand_ops.h): prand_dev::Gen<GEN>::skipahead(ops, s)
 *   advances a stream by s * dist for any s < 2^levels.  The table is owned by `st` and stays valid until
 *   the next prand_device_ops call on `st` or prand_free.  1 <= levels <= 64.  Synchronises the stream.
 *
 * prand_device_api_init_fill_{u32,f32,f64} -- the library's example kernel for that path: `st` holds ONE
 *   stream (the base stream, else PRAND_ERR_ARG); every stream s < n_streams is initialised on the device
 *   (base stream loaded, skipped s * block_len ahead with the table) and generates n_per_stream numbers
 *   into out[i * n_streams + s] -- exactly the numbers of prand_init(..., n_streams, block_len) +
 *   prand_generate_*.  MT19937 runs one CTA per stream (CTA-cooperative skip, warp-cooperative generator).
 *   The base state is not modified.
 */
int prand_device_ops(prand_state *st, uint64_t dist_mant, unsigned dist_log2, unsigned levels,
                     const void **d_ops, void *cuda_stream);
int prand_device_api_init_fill_u32(prand_state *st, uint64_t block_len_mant, unsigned block_len_log2,
                                   uint64_t n_streams, uint32_t *out, uint64_t n_per_stream, void *cuda_stream);
int prand_device_api_init_fill_f32(prand_state *st, uint64_t block_len_mant, unsigned block_len_log2,
                                   uint64_t n_streams, float *out, uint64_t n_per_stream, void *cuda_stream);
int prand_device_api_init_fill_f64(prand_state *st, uint64_t block_len_mant, unsigned block_len_log2,
                                   uint64_t n_streams, double *out, uint64_t n_per_stream, void *cuda_stream);

void *prand_state_device_ptr(prand_state *st);
uint64_t prand_state_n_streams(const prand_state *st);
int prand_device_api_fill_u32(prand_state *st, uint32_t *out, uint64_t n_per_stream, void *cuda_stream);
int prand_device_api_fill_f32(prand_state *st, float *out, uint64_t n_per_stream, void *cuda_stream);
int prand_device_api_fill_f64(prand_state *st, double *out, uint64_t n_per_stream, void *cuda_stream);

/*
 * Canonical state export / import (the state is plain data and may be copied between
 * host and device; generation continues from it).  Per stream, little-endian, streams consecutive:
 *   LFSR113   4 x u32  z1..z4 masked to their significant top 31/29/28/25 bits;
 *   MRG32K3A  6 x u32  x_n, x_{n-1}, x_{n-2}, y_n, y_{n-1}, y_{n-2};
 *   MT19937   624 x u32 window x_P..x_{P+623}, low 31 bits of word 0 zeroed;
 *   GM/GQ     2s words xP_0, xN_0, ..., xP_{s-1}, xN_{s-1} (u32 if g < 2^32, else u64), residues mod g.
 * prand_state_bytes() = n_streams * per-stream bytes.  Both calls synchronise the device.
 * prand_set_state checks the words: LFSR113 components with all significant bits zero, MRG32K3A words that are
 * not residues mod m1 / m2 or a component that is all zero, and GM/GQ words >= g are refused (PRAND_ERR_ARG,
 * nothing is changed).
 */
size_t prand_state_bytes(const prand_state *st);
int prand_get_state(const prand_state *st, void *host_buf, size_t bytes);
int prand_set_state(prand_state *st, const void *host_buf, size_t bytes);

uint64_t prand_n_streams(const prand_state *st);
int prand_gen_of(const prand_state *st);

/*
 * Releases the state and every device buffer it owns.  The release is STREAM-ORDERED on the CUDA stream of
 * the state's most recent call (no device synchronisation): work queued there before prand_free still sees
 * the buffers; the caller must not have work on OTHER streams that still uses the state or the pointer of
 * prand_state_device_ptr / prand_device_ops.
 */
int prand_free(prand_state *st);

/*
 * Device memory comes from a stream-ordered pool owned by the library (one per device, never shrunk, so that
 * prand_init + prand_free cost microseconds).  prand_trim returns the pool's unused memory of the current
 * device to the driver; call it after freeing large states if other allocators need the memory.
 */
int prand_trim(void);

/* MT19937: the generation kernels address a row block with 32-bit byte offsets; prand_init refuses more streams
 * per state (PRAND_ERR_ARG).  2.58 million streams = 6.4 GB of state; shard larger families (prand_init_shard). */
#define PRAND_MT19937_MAX_STREAMS 2581102ull

/*
 * prand_fill_u32 -- write-peak probe: 128-bit stores of a constant to `n_words` u32 at device
 *   pointer `out` (16-byte aligned).  Used by the bench to measure the HBM write roofline in the
 *   same run as the generators.
 */
int prand_fill_u32(uint32_t *out, uint64_t n_words, uint32_t value, void *cuda_stream);

/*
 * Measurement probes; none of them is on the hot path.
 *   prand_probe_empty   launches an empty kernel (1 CTA x 32 threads) on `cuda_stream`: the launch floor
 *                       that small configurations (C1) are compared with.
 *   prand_probe_memset  cudaMemsetAsync of `bytes` at DEVICE pointer d_ptr: second opinion on the write peak.
 *   prand_probe_pipe    launches the instruction-rate probe number `op` (0 .. prand_probe_pipe_count()-1,
 *                       named by prand_probe_pipe_name) on 8 CTAs x 256 threads per SM; *thread_ops (HOST
 *                       pointer) receives the thread-level operations one launch executes, so that
 *                       thread_ops / (time x SM clock x SM count) = operations per clock per SM
 *                       (profiles/pipe_rates.md).
 */
int prand_probe_empty(void *cuda_stream);
int prand_probe_memset(void *d_ptr, int value, size_t bytes, void *cuda_stream);
int prand_probe_pipe_count(void);
const char *prand_probe_pipe_name(int op);
int prand_probe_pipe(int op, uint64_t iters, uint64_t *thread_ops, void *cuda_stream);

/*
 * prand_debug_set -- test / tuning hooks that select alternate kernels or algorithms; results never
 *   change.  The hooks live in one process-wide table that is filled once from the environment
 *   variables of the same names when the library first needs it; this call changes one entry afterwards
 *   (value NULL or "" restores the default).  Names: PRAND_MT_CFG (0..6: MT19937 generation kernel),
 *   PRAND_MT_APPLY (list, win, win2, win4, multi: other polynomial-application kernels), PRAND_GM_LP (1, 2, 4), PRAND_GM31_NF (0, 10, 12, 14, 16), PRAND_GM_WATCH,
 *   PRAND_MRG_INT, PRAND_GM_INIT (matrix), PRAND_CHUNK_LEN, PRAND_LFSR_INIT (table: the paper's 128-table
 *   jump), PRAND_MT_POLY (host: no precomputed polynomial table), PRAND_SEQ_SECTIONS (cap on the sections
 *   of prand_generate_seq_*; not MT19937).  Unknown name:
 *   PRAND_ERR_ARG.  The launch paths read the table without a lock: call this only while no other thread is inside a
 *   libprand call (it is a test and tuning aid, not a run-time switch).
 */
int prand_debug_set(const char *name, const char *value);

/* Number of kernels this library has launched in this process (for bench.py's gpu_launches). */
uint64_t prand_launch_count(void);

/* Bytes of prepared operator tables / seed states this library has copied host-to-device so far. */
uint64_t prand_uploaded_bytes(void);

/* Name of the kernel configuration the last generate call on `st` used (static string). */
const char *prand_last_kernel(const prand_state *st);

const char *prand_strerror(int code);
/* cudaError_t of the last failing CUDA call in this thread (0 if none). */
int prand_last_cuda_error(void);
const char *prand_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PRAND_H */
