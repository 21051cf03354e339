// k_noalloc.cu -- prand_lfsr113_seq_noalloc_u32: the single-sequence fill for callers that must not allocate.
//
// Who this is for.  Every other generating call of libprand needs a prand_state, and prand_init takes the
// state's device memory from the library's stream-ordered pool; prand_generate_seq_* additionally keeps a table of
// section start states (and, for some generators, a scratch copy of the output) that it allocates on demand.  Some
// users cannot make such calls at the point where they need random numbers:
//   * code that runs inside a region where the CUDA allocator must not be touched -- a latency-critical loop whose
//     memory was carved out of one arena at start-up, a framework whose caching allocator owns the whole device and
//     forbids foreign cudaMalloc / pool growth, a process close to its memory limit where an allocation may fail or
//     trigger a device-wide synchronisation;
//   * plug-ins and callbacks that are handed device buffers by their host application and are not allowed to
//     create any of their own.
// For them this file provides ONE entry point that allocates and frees nothing on the device: the caller passes the
// generator state (16 bytes of its own device memory) and the output array; the table of section start states and
// the jump operators -- the scratch memory the sectioned fill needs ("the output array is divided
// into sections ... jumping ahead to a starting point of the section") -- live in a fixed array that is part of the
// library image.
//
// The scratch array.  `g_noalloc_scratch` below is a file-scope __device__ array of NOALLOC_SCRATCH_BYTES (520 KiB).
// Every GPU on which the library is loaded holds a copy from module load until the process exits, whether or not
// this entry point is ever called; that is the price of not allocating, and the reason the capacity is modest
// (PRAND_NOALLOC_MAX_LENGTH numbers per call; longer arrays are filled by several calls, the state carries on).
// Inside host code the name `g_noalloc_scratch` is only a host-side handle of the symbol, not a device address
// (a kernel given it would fault, or on systems where the GPU can reach host memory silently use the wrong bytes),
// so the host asks the runtime for the array's address on the current device with cudaGetSymbolAddress -- once per
// device, see scratch_of() -- and passes that pointer to the kernels.
//
// Sharing.  All calls on one device use the same array and find in it whatever the previous call left.  Nothing
// in it has to start from zero: a call first writes the operators and section states it is going to read (words
// beyond the sections of this call are stale and never read).  Two calls whose GPU work overlaps -- different CUDA
// streams without an ordering between them, or different host threads -- race on the array and produce garbage;
// callers serialise them (one stream, or events).
//
// Product code: shares nothing with oracle/.
#include <mutex>
#include <vector>
#include "internal.h"
#include "skip_ops.h"
#include "../../include/prand_device.cuh"

using namespace prand;

namespace {

constexpr uint64_t MAX_SECTIONS = PRAND_NOALLOC_MAX_SECTIONS;            // section start states the array holds
constexpr unsigned SECTION_LEVELS = 15;                                  // operators L 2^j reach section 2^15 - 1
constexpr unsigned OP_SLOTS = SECTION_LEVELS + 1;                        // + the operator of distance `length`
constexpr size_t OPS_BYTES = OP_SLOTS * sizeof(LfsrOp);                  // 8 KiB
constexpr size_t STATES_BYTES = 4 * MAX_SECTIONS * sizeof(uint32_t);     // 512 KiB, structure of arrays z[c][section]
constexpr size_t NOALLOC_SCRATCH_BYTES = OPS_BYTES + STATES_BYTES;
static_assert((MAX_SECTIONS & (MAX_SECTIONS - 1)) == 0 && MAX_SECTIONS == (1ull << SECTION_LEVELS),
              "the level count is the bit length of the largest section index");
static_assert(OPS_BYTES % 256 == 0, "the state table starts on a 256-byte boundary");

// The scratch memory itself.  Host code must not pass this name to a kernel: see scratch_of().
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

// Device address of g_noalloc_scratch on the CURRENT device, looked up once per device (with that device current)
// and remembered.  cudaGetSymbolAddress may load the module on this device the first time, which is why the first
// call on a device should not happen inside a stream capture.
cudaError_t scratch_of(unsigned char **p)
{
    static std::mutex mu;
    static unsigned char *per_device[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!per_device[dev]) {
        unsigned char *d = nullptr;
        e = cudaGetSymbolAddress((void **)&d, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!d) return cudaErrorInvalidSymbol;
        per_device[dev] = d;
    }
    *p = per_device[dev];
    return cudaSuccess;
}

// The caller's state moves on by the distance of `op` and is left in the canonical form of prand_get_state (only
// the top 31 / 29 / 28 / 25 bits of a component are state, reading L3 of DESIGN.md; the rest is cleared).
__global__ void lfsr113_advance_canonical_kernel(uint32_t *state, const LfsrOp *__restrict__ op)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    uint32_t z[4];
    for (int c = 0; c < 4; c++) z[c] = state[c];
    prand_dev::lfsr113_apply_bits(op, 1, z);
    const uint32_t significant[4] = {0xFFFFFFFEu, 0xFFFFFFF8u, 0xFFFFFFF0u, 0xFFFFFF80u};
    for (int c = 0; c < 4; c++) state[c] = z[c] & significant[c];
}

}  // namespace

#define NA_CU(call)                                                  \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return prand::record_cuda_error(e_);  \
    } while (0)

extern "C" int prand_lfsr113_seq_noalloc_u32(uint32_t *d_state, uint32_t *out, uint64_t length, void *cuda_stream)
{
    if (!d_state || (uintptr_t)d_state % 4) return PRAND_ERR_ARG;
    if (length == 0) return PRAND_OK;
    if (!out || (uintptr_t)out % 16) return PRAND_ERR_ARG;
    if (length > PRAND_NOALLOC_MAX_LENGTH) return PRAND_ERR_CAPACITY;
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    // section plan (Table 5): sections of at least 1024 numbers, at most MAX_SECTIONS of them,
    // section length a multiple of 32 (the fill kernel writes 32-row blocks); the last section may be shorter
    uint64_t S = length / 1024;
    if (S > MAX_SECTIONS) S = MAX_SECTIONS;
    if (S < 1) S = 1;
    uint64_t L = (length + S - 1) / S;
    L = (L + 31) / 32 * 32;
    S = (length + L - 1) / L;

    // step a0 on the host: the operators of distance L 2^j for the bits of a section index, and of `length`
    unsigned levels = 0;
    while (levels < 64 && ((S - 1) >> levels)) levels++;
    if (levels > SECTION_LEVELS) return PRAND_ERR_INTERNAL;
    std::vector<LfsrOp> ops, adv;
    host::lfsr113_levels(host::Dist{L, 0}, levels, ops);
    host::lfsr113_levels(host::Dist{length, 0}, 1, adv);
    if (ops.size() != levels || adv.size() != 1) return PRAND_ERR_INTERNAL;

    unsigned char *scratch = nullptr;
    NA_CU(scratch_of(&scratch));
    LfsrOp *d_ops = (LfsrOp *)scratch;
    uint32_t *d_sections = (uint32_t *)(scratch + OPS_BYTES);
    // (pageable source: the runtime has taken its copy of the bytes when cudaMemcpyAsync returns)
    if (levels) NA_CU(cudaMemcpyAsync(d_ops, ops.data(), levels * sizeof(LfsrOp), cudaMemcpyHostToDevice, stream));
    NA_CU(cudaMemcpyAsync(d_ops + SECTION_LEVELS, adv.data(), sizeof(LfsrOp), cudaMemcpyHostToDevice, stream));

    LaunchInfo li;
    // section c starts c * L numbers ahead of the caller's state: written to the static table
    JumpArgs a = {};
    a.base = d_state;
    a.st_in = nullptr;
    a.st_out = d_sections;
    a.n_streams = S;
    a.ops = d_ops;
    a.idx0 = 0;
    a.idx_stride = 1;
    NA_CU(lfsr113_jump(stream, a, &li));
    prand::count_launches(li.launches);
    // one thread per section reads its start state from the table and writes its numbers in place
    NA_CU(lfsr113_seq(stream, d_sections, out, DT_U32, S, L, length, &li));
    prand::count_launches(li.launches);
    // the caller's state moves on by `length` (after the section table has been derived from it: stream order)
    lfsr113_advance_canonical_kernel<<<1, 32, 0, stream>>>(d_state, d_ops + SECTION_LEVELS);
    NA_CU(cudaGetLastError());
    prand::count_launches(1);
    return PRAND_OK;
}
