// internal.h -- types shared by the host-side preparation (prand.cu) and the kernel files.
// Product code: shares nothing with oracle/.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/prand.h"
#include "../../include/prand_ops.h"

namespace prand {

enum { DT_U32 = 0, DT_F32 = 1, DT_F64 = 2 };

// ---- skip operators (a0 builds them on the host, the kernels apply them): include/prand_ops.h --------
typedef prand_lfsr113_op LfsrOp;
typedef prand_mrg32k3a_op MrgOp;
typedef prand_gm_op GmOp;
typedef prand_mt19937_op MtOp;

// GM/GQ parameters, Table 2 + Table 5 ensemble sizes.
struct GmParams {
    uint64_t k, q, g;
    unsigned v, s, d;      // output bits per point, ensemble size, log2 of the orbit spacing D
    unsigned nbits;        // bit length of g
    uint64_t mu;           // floor(2^(2 nbits) / g) for Barrett reduction in the jump kernels
    bool wide;             // state words are u64 (g >= 2^32)
};
const GmParams *gm_params(int gen);   // nullptr if gen is not a GM/GQ generator

// How a jump kernel finds the exponent of stream j: idx = idx0 + j * idx_stride; the operator
// applied is prod_{bit b of idx set} ops[b].  base != nullptr: start from the broadcast base state
// instead of st_in (stream initialisation).
struct JumpArgs {
    const void *base;
    const void *st_in;
    void *st_out;
    uint64_t n_streams;
    const void *ops;       // device array of per-level operators
    uint64_t idx0, idx_stride;
    uint64_t count;        // streams to compute (the first `count` of n_streams; 0 = all): GM tree init
};

// One bulk generation launch.  Rows [0, n) of every stream; when n_chunks > 1 virtual stream
// (s, c) first jumps c * chunk_len ahead with chunk_ops[c - 1] (the operator of distance
// c * chunk_len, c = 1..n_chunks-1) and fills rows [c*chunk_len, min(n, (c+1)*chunk_len)); the last
// chunk writes the final state to st_out.
struct GenArgs {
    const void *st_in;
    void *st_out;
    void *out;
    int dtype;
    uint64_t n_streams;
    uint64_t n;
    uint64_t chunk_len;
    uint64_t n_chunks;
    const void *chunk_ops;
    bool clean;            // GM55/GQ58: every state word is a multiple of 2^t (see k_gmgq.cu)
};

struct LaunchInfo { const char *kernel; unsigned launches; };

cudaError_t lfsr113_jump(cudaStream_t, const JumpArgs &, LaunchInfo *);
// the paper's 128-table method: stream j advanced (idx0 + j * idx_stride) * mant * 2^log2,
// one warp per stream; a.ops is not used
cudaError_t lfsr113_table_jump(cudaStream_t, const JumpArgs &, uint64_t mant, unsigned log2, LaunchInfo *);
cudaError_t lfsr113_generate(cudaStream_t, const GenArgs &, LaunchInfo *);
// sections of one sequence in PRAND's contiguous layout out[c * sec_len + i] (sec_len a multiple of 32, out 16-byte
// aligned); st_in = the section family's state (structure of arrays); the caller advances the sequence's own state
cudaError_t lfsr113_seq(cudaStream_t, const void *st_in, void *out, int dtype, uint64_t n_sections, uint64_t sec_len,
                        uint64_t length, LaunchInfo *);
// small outputs (they stay in L2) from few streams: one stream per thread, so that four times as many threads share
// the work and a sub-section's jump is paid once per 64 rows of one stream instead of four (C1: 18 -> 14 us)
inline bool lfsr113_narrow(uint64_t ns, uint64_t n, int dtype, int sms)
{
    const uint64_t esz = dtype == DT_F64 ? 8 : 4;
    return 2 * ns <= (uint64_t)sms * 1024 && ns * n * esz <= (64ull << 20);
}
cudaError_t mrg32k3a_jump(cudaStream_t, const JumpArgs &, LaunchInfo *);
cudaError_t mrg32k3a_generate(cudaStream_t, const GenArgs &, LaunchInfo *);
// sections of one sequence written in PRAND's contiguous layout (sec_len a multiple of 16, out 16-byte aligned);
// st_last (one stream) receives the state of the sequence after `length` numbers
cudaError_t mrg32k3a_seq_f64(cudaStream_t, const void *st_in, void *st_last, double *out, uint64_t n_sections,
                             uint64_t sec_len, uint64_t length, LaunchInfo *);
// the same layout for u32 / f32 outputs (sec_len a multiple of 32); the caller advances the sequence's own state
cudaError_t mrg32k3a_seq4(cudaStream_t, const void *st_in, void *out, int dtype, uint64_t n_sections, uint64_t sec_len,
                          uint64_t length, LaunchInfo *);
cudaError_t gm_jump(cudaStream_t, int gen, const JumpArgs &, LaunchInfo *);
cudaError_t gm_generate(cudaStream_t, int gen, const GenArgs &, LaunchInfo *);
// streams [s_begin, s_end) = kn * stream(s - back) - qn * stream(s - 2 back) (eq. 2), in place
cudaError_t gm_tree_fill(cudaStream_t, int gen, void *st, uint64_t ns, uint64_t s_begin, uint64_t s_end,
                         uint64_t back, uint64_t kn, uint64_t qn, LaunchInfo *);
// MT19937: dst stream j (j in [dst0, dst0+count)) = g(A) applied to src stream (j - src_back), or to
// itself when src_back == 0.  State layout [stream][624].
// h_op: the same polynomial in host memory if the caller has it (it then travels as a kernel argument), else nullptr
cudaError_t mt19937_apply(cudaStream_t, const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                          uint64_t count, uint64_t src_back, const MtOp *d_op, const MtOp *h_op, LaunchInfo *);
cudaError_t mt19937_generate(cudaStream_t, const GenArgs &, LaunchInfo *);
// sections of one sequence in PRAND's contiguous layout out[c * sec_len + i] (sec_len even, out 16-byte aligned);
// st_in = [n_sections][624] windows, st_last (one window) receives the state after `length` numbers
cudaError_t mt19937_seq(cudaStream_t, const void *st_in, void *st_last, void *out, int dtype, uint64_t n_sections,
                        uint64_t sec_len, uint64_t length, LaunchInfo *);
cudaError_t fill_u32(cudaStream_t, uint32_t *out, uint64_t n_words, uint32_t value, LaunchInfo *);
// out[c * sec_len + i] = tmp[i * n_sections + c] for c * sec_len + i < length (elem_bytes 4 or 8)
cudaError_t transpose_sections(cudaStream_t, const void *tmp, void *out, uint64_t n_sections, uint64_t sec_len,
                               uint64_t length, int elem_bytes, LaunchInfo *);

// one thread per stream through include/prand_device.cuh (example / self-test of the device API)
cudaError_t devapi_generate(cudaStream_t, int gen, void *state, void *out, uint64_t ns, uint64_t n, int dtype,
                            LaunchInfo *);

// device-side stream initialisation example: stream s = base stream skipped s * dist ahead with the table `ops`
cudaError_t devapi_init_generate(cudaStream_t, int gen, const void *base, const void *ops, void *out, uint64_t ns,
                                 uint64_t n, int dtype, LaunchInfo *);

int sm_count();   // multiprocessor count of the current device

// for entry points that live outside prand.cu: remember a failed CUDA call for prand_last_cuda_error (returns
// PRAND_ERR_CUDA), add to the count behind prand_launch_count
int record_cuda_error(cudaError_t e);
void count_launches(unsigned n);

// Test / tuning hooks.  One process-wide struct, filled ONCE from the PRAND_* environment variables the
// first time the library needs it and changed afterwards only through prand_debug_set (prand.h): the
// launch paths read plain fields, never the environment.
struct DebugHooks {
    int mt_cfg;             // PRAND_MT_CFG: force an MT19937 generation kernel variant (-1: by stream count)
    bool mt_apply_list;     // PRAND_MT_APPLY=list: the position-list application kernel at any size
    bool mt_apply_win;      // PRAND_MT_APPLY=win | win2 | win4: the one-stream-per-CTA window kernel (1, 2 or 4 slices of
                            // 160 threads) at any size, instead of the forms chosen by the number of applications
    int mt_apply_nsl;
    int gm_lp;              // PRAND_GM_LP: lanes per GM61 stream (0: default)
    int gm31_nf;            // PRAND_GM31_NF: GM31 points on the FP64 pipe (-1: default 14)
    bool gm_watch_set;      // PRAND_GM_WATCH: limit of the optimistic steps' watch value
    uint32_t gm_watch;
    bool mrg_int;           // PRAND_MRG_INT: all-integer MRG32K3A kernel for 4-byte outputs
    bool gm_init_matrix;    // PRAND_GM_INIT=matrix: one matrix jump per stream instead of the eq.-2 tree
    uint64_t chunk_len;     // PRAND_CHUNK_LEN: force the sub-section length (0: plan_chunks decides)
    bool lfsr_table;        // PRAND_LFSR_INIT=table: the paper's 128-table jump method for LFSR113
    bool mt_host_poly;      // PRAND_MT_POLY=host: compute every MT19937 jump polynomial on the host (no table)
    uint64_t seq_sections;  // PRAND_SEQ_SECTIONS: cap on the sections of prand_generate_seq_* (0: the plan's own, 2^17)
};
const DebugHooks &debug_hooks();

}  // namespace prand
