// prand.cu -- the C-ABI boundary of libprand (include/prand.h, include/prand_host.h): argument
// checks, host preparation of the skip operators (a0, skip_ops.cpp), state management, launch policy
// and the calls into the kernel files.  Every arithmetic step of the hot path runs in the kernels;
// there is no CPU fallback.  Product code: shares nothing with oracle/.
#include <atomic>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>
#include "internal.h"
#include "skip_ops.h"
#include "../../include/prand_host.h"

using namespace prand;
using prand::host::Dist;

// ---- generator tables -----------------------------------------------------------------------------
namespace prand {

static GmParams make_gm(uint64_t k, uint64_t q, uint64_t g, unsigned v, unsigned s, unsigned d)
{
    GmParams p;
    p.k = k; p.q = q; p.g = g; p.v = v; p.s = s; p.d = d;
    p.nbits = 64 - (unsigned)__builtin_clzll(g);
    p.mu = (uint64_t)((((unsigned __int128)1) << (2 * p.nbits)) / g);
    p.wide = g >= (1ull << 32);
    return p;
}

// Table 2: k, q, g, v; Table 5: ensemble size s; d: reading G3.
const GmParams *gm_params(int gen)
{
    static const GmParams tab[8] = {
        make_gm(15, 28, (1ull << 19) - 1, 1, 32, 32),                          // GM19
        make_gm(4, 2, (1ull << 29) - 3, 1, 32, 52),                            // GM29
        make_gm(11, 14, (1ull << 31) - 1, 1, 32, 56),                          // GM31
        make_gm(256, 176, 16ull * ((1ull << 51) - 129), 4, 8, 98),             // GM55
        make_gm(24, 74, (1ull << 61) - 1, 1, 32, 116),                         // GM61
        make_gm(8, 48, ((1ull << 29) - 3) << 29, 1, 32, 52),                   // GQ58.1
        make_gm(8, 48, ((1ull << 29) - 3) << 29, 3, 12, 54),                   // GQ58.3
        make_gm(8, 48, ((1ull << 29) - 3) << 29, 4, 8, 54),                    // GQ58.4
    };
    if (gen < PRAND_GM19 || gen > PRAND_GQ58_4) return nullptr;
    return &tab[gen - PRAND_GM19];
}

int sm_count()
{
    // per device, no shared mutable cache: the attribute query costs well under a microsecond
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    return n;
}

namespace {
std::mutex g_hooks_mu;
DebugHooks g_hooks;
std::once_flag g_hooks_once;

void hook_assign(DebugHooks &h, const std::string &name, const char *v)
{
    const bool on = v && *v;
    if (name == "PRAND_MT_CFG") h.mt_cfg = on ? std::atoi(v) : -1;
    else if (name == "PRAND_MT_APPLY") {
        const std::string m = on ? v : "";
        h.mt_apply_list = m == "list";
        h.mt_apply_nsl = m == "win" ? 1 : m == "win2" ? 2 : m == "win4" ? 4 : m == "multi" ? -1 : 0;
        h.mt_apply_win = h.mt_apply_nsl > 0;
    }
    else if (name == "PRAND_GM_LP") h.gm_lp = on ? std::atoi(v) : 0;
    else if (name == "PRAND_GM31_NF") h.gm31_nf = on ? std::atoi(v) : -1;
    else if (name == "PRAND_GM_WATCH") { h.gm_watch_set = on; h.gm_watch = on ? (uint32_t)std::strtoul(v, nullptr, 0) : 0; }
    else if (name == "PRAND_MRG_INT") h.mrg_int = on;
    else if (name == "PRAND_GM_INIT") h.gm_init_matrix = on && std::string(v) == "matrix";
    else if (name == "PRAND_CHUNK_LEN") h.chunk_len = on ? std::strtoull(v, nullptr, 10) : 0;
    else if (name == "PRAND_LFSR_INIT") h.lfsr_table = on && std::string(v) == "table";
    else if (name == "PRAND_MT_POLY") h.mt_host_poly = on && std::string(v) == "host";
    else if (name == "PRAND_SEQ_SECTIONS") h.seq_sections = on ? std::strtoull(v, nullptr, 10) : 0;
}
const char *const HOOK_NAMES[] = {"PRAND_MT_CFG", "PRAND_MT_APPLY", "PRAND_GM_LP", "PRAND_GM31_NF", "PRAND_GM_WATCH",
                                  "PRAND_MRG_INT", "PRAND_GM_INIT", "PRAND_CHUNK_LEN", "PRAND_LFSR_INIT", "PRAND_MT_POLY",
                                  "PRAND_SEQ_SECTIONS"};
void hooks_from_env()
{
    for (const char *n : HOOK_NAMES) hook_assign(g_hooks, n, std::getenv(n));
}
}  // namespace

const DebugHooks &debug_hooks()
{
    std::call_once(g_hooks_once, hooks_from_env);
    return g_hooks;
}

}  // namespace prand

namespace {

std::atomic<uint64_t> g_launches{0};
std::atomic<uint64_t> g_h2d_bytes{0};   // operator tables and seed states uploaded by init/jump/generate
thread_local int g_last_cuda_error = 0;

inline bool is_gm(int gen) { return gen >= PRAND_GM19 && gen <= PRAND_GQ58_4; }

// words per stream and bytes per word of the state (internal SoA and canonical export agree on both)
inline size_t state_words(int gen)
{
    if (gen == PRAND_LFSR113) return 4;
    if (gen == PRAND_MRG32K3A) return 6;
    if (gen == PRAND_MT19937) return host::MT_N;
    if (const GmParams *p = gm_params(gen)) return 2 * (size_t)p->s;
    return 0;
}
inline size_t state_word_bytes(int gen)
{
    const GmParams *p = gm_params(gen);
    return (p && p->wide) ? 8 : 4;
}
inline size_t stream_bytes(int gen) { return state_words(gen) * state_word_bytes(gen); }

inline unsigned bit_length(uint64_t x) { return x ? 64u - (unsigned)__builtin_clzll(x) : 0u; }

int cuda_fail(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    return PRAND_ERR_CUDA;
}
// host-to-device upload of a prepared table, counted for bench.py's h2d_bytes_per_step
#define UPLOAD(dst, src, bytes, stream)                                                        \
    do {                                                                                       \
        CU(cudaMemcpyAsync((dst), (src), (bytes), cudaMemcpyHostToDevice, (stream)));          \
        g_h2d_bytes.fetch_add((bytes), std::memory_order_relaxed);                             \
    } while (0)
#define CU(call)                                         \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) return cuda_fail(e_);     \
    } while (0)

// Device memory comes from the stream-ordered allocator, from a pool of the library's own (one per device,
// release threshold "never": init / free of a state cost microseconds and never synchronise the device, so
// that prand_init + prand_generate + prand_free can be a hot loop).  The process's default pool is left
// alone; prand_trim() hands the cached memory back to the driver.
std::mutex g_pool_mu;
cudaMemPool_t g_pools[64] = {};
cudaError_t device_pool(cudaMemPool_t *pool)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t p;
        e = cudaMemPoolCreate(&p, &props);
        if (e != cudaSuccess) return e;
        uint64_t keep = UINT64_MAX;
        e = cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) { cudaMemPoolDestroy(p); return e; }
        g_pools[dev] = p;
    }
    *pool = g_pools[dev];
    return cudaSuccess;
}
cudaError_t dev_alloc(void **p, size_t bytes, cudaStream_t stream)
{
    cudaMemPool_t pool;
    cudaError_t e = device_pool(&pool);
    if (e != cudaSuccess) return e;
    return cudaMallocFromPoolAsync(p, bytes ? bytes : 1, pool, stream);
}

}  // namespace

namespace {
// the precomputed MT19937 polynomials, resident in device memory (one copy per device, uploaded
// the first time a jump of a tabulated form needs them; 4.5 MB).  Record layout = MtOp (624 u32 words).
const MtOp *mt_device_table(cudaStream_t stream)
{
    static std::mutex mu;
    static const MtOp *per_device[64] = {};
    const host::MtPoly *t = host::mt19937_table();
    int dev = 0;
    if (!t || cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (!per_device[dev]) {
        void *d = nullptr;
        const size_t bytes = (size_t)host::MT_TABLE_ENTRIES * sizeof(MtOp);
        static_assert(sizeof(MtOp) == sizeof(host::MtPoly), "table records are uploaded as they are");
        if (cudaMalloc(&d, bytes) != cudaSuccess) return nullptr;
        if (cudaMemcpyAsync(d, t, bytes, cudaMemcpyHostToDevice, stream) != cudaSuccess ||
            cudaStreamSynchronize(stream) != cudaSuccess) { cudaFree(d); return nullptr; }
        g_h2d_bytes.fetch_add(bytes, std::memory_order_relaxed);
        per_device[dev] = (const MtOp *)d;
    }
    return per_device[dev];
}
}  // namespace

struct prand_state {
    int gen;
    int device;
    uint64_t ns;            // streams held by this state
    uint64_t first;         // global index of local stream 0
    void *d_state[2];       // [cur] holds the streams; the other one is the target of chunked launches
    int cur;
    size_t bytes;           // ns * stream_bytes(gen)
    void *d_ops;            // scratch for uploaded operator tables (grown on demand)
    size_t ops_bytes;
    void *d_chunk_ops;      // cached operators for chunk_len * 2^j
    uint64_t chunk_len;
    uint64_t chunk_count;   // operators cached for c = 1..chunk_count-1
    void *d_stage[2];       // device staging of the *_host calls
    size_t stage_bytes;
    cudaStream_t copy_stream;
    cudaEvent_t ev_gen[2], ev_copy[2];
    bool host_ready;
    const char *last_kernel;
    cudaStream_t last_stream;   // stream of the most recent call: prand_free releases in its order
    void *d_user_ops;       // prand_device_ops: operator table handed to the caller's kernels
    prand_state *sec;       // prand_generate_seq_*: cached family of sections (one stream per section)
    bool gm_clean;          // GM55/GQ58: every state word is a multiple of 2^t (true for states the
                            // library creates; an imported state is scanned), see k_gmgq.cu
};

namespace {

int ensure_ops(prand_state *st, size_t bytes)
{
    if (bytes <= st->ops_bytes) return PRAND_OK;
    if (st->d_ops) { CU(cudaFreeAsync(st->d_ops, st->last_stream)); st->d_ops = nullptr; st->ops_bytes = 0; }
    CU(dev_alloc(&st->d_ops, bytes, st->last_stream));
    st->ops_bytes = bytes;
    return PRAND_OK;
}

int ensure_second_buffer(prand_state *st)
{
    if (st->d_state[1 - st->cur]) return PRAND_OK;
    CU(dev_alloc(&st->d_state[1 - st->cur], st->bytes, st->last_stream));
    return PRAND_OK;
}

void note(prand_state *st, const LaunchInfo &li)
{
    g_launches.fetch_add(li.launches, std::memory_order_relaxed);
    if (st) st->last_kernel = li.kernel;
}

// Host operators for distance n * 2^j, j < levels, as a flat byte vector in the kernels' layout.
int build_level_ops(int gen, Dist n, unsigned levels, std::vector<unsigned char> &bytes)
{
    if (gen == PRAND_LFSR113) {
        std::vector<LfsrOp> v;
        host::lfsr113_levels(n, levels, v);
        bytes.assign((unsigned char *)v.data(), (unsigned char *)(v.data() + v.size()));
    } else if (gen == PRAND_MRG32K3A) {
        std::vector<MrgOp> v;
        host::mrg32k3a_levels(n, levels, v);
        bytes.assign((unsigned char *)v.data(), (unsigned char *)(v.data() + v.size()));
    } else if (is_gm(gen)) {
        std::vector<GmOp> v;
        host::gm_levels(*gm_params(gen), n, levels, v);
        bytes.assign((unsigned char *)v.data(), (unsigned char *)(v.data() + v.size()));
    } else if (gen == PRAND_MT19937) {
        std::vector<host::MtPoly> v;
        host::mt19937_levels(n, levels, v);
        std::vector<MtOp> ops(v.size());
        for (size_t i = 0; i < v.size(); i++) host::mt19937_to_op(v[i], ops[i]);
        bytes.assign((unsigned char *)ops.data(), (unsigned char *)(ops.data() + ops.size()));
    } else {
        return PRAND_ERR_GEN;
    }
    return PRAND_OK;
}

// Canonical seed state of one stream (not masked), words of state_word_bytes(gen).
int build_seed_state(int gen, uint64_t seed, std::vector<unsigned char> &bytes)
{
    bytes.assign(stream_bytes(gen), 0);
    if (gen == PRAND_LFSR113) {
        // all four words = seed; a component whose significant top bits vanish stays zero forever
        if (seed > 0xFFFFFFFFull || (seed & 0xFFFFFF80ull) == 0) return PRAND_ERR_SEED;
        uint32_t *w = (uint32_t *)bytes.data();
        for (int c = 0; c < 4; c++) w[c] = (uint32_t)seed;
    } else if (gen == PRAND_MRG32K3A) {
        if (seed == 0 || seed >= 4294944443ull) return PRAND_ERR_SEED;
        uint32_t *w = (uint32_t *)bytes.data();
        for (int c = 0; c < 6; c++) w[c] = (uint32_t)seed;
    } else if (gen == PRAND_MT19937) {
        if (seed > 0xFFFFFFFFull) return PRAND_ERR_SEED;
        host::mt19937_seed_state((uint32_t)seed, (uint32_t *)bytes.data());
    } else if (const GmParams *p = gm_params(gen)) {
        uint64_t words[64];
        if (!host::gm_seed_state(*p, seed, words)) return PRAND_ERR_SEED;
        for (unsigned i = 0; i < 2 * p->s; i++) {
            if (p->wide) ((uint64_t *)bytes.data())[i] = words[i];
            else ((uint32_t *)bytes.data())[i] = (uint32_t)words[i];
        }
    } else {
        return PRAND_ERR_GEN;
    }
    return PRAND_OK;
}

// dist != nullptr: the distance the level-0 operator of a.ops stands for (the LFSR113 table method works
// from the distance itself)
cudaError_t launch_jump(cudaStream_t stream, int gen, const JumpArgs &a, LaunchInfo *li, const Dist *dist = nullptr)
{
    if (gen == PRAND_LFSR113 && dist && debug_hooks().lfsr_table)
        return lfsr113_table_jump(stream, a, dist->mant, dist->log2, li);
    if (gen == PRAND_LFSR113) return lfsr113_jump(stream, a, li);
    if (gen == PRAND_MRG32K3A) return mrg32k3a_jump(stream, a, li);
    return gm_jump(stream, gen, a, li);
}

}  // namespace

// ==================================================================================================
// prand_init / prand_init_shard (a0 + a1)
// ==================================================================================================
namespace {

// MT19937: stream 0 of the shard = seed window jumped first * L; then a doubling tree -- level j
// fills local streams [2^j, 2^(j+1)) from [0, 2^j) with g_{L 2^j} (eq. 10), one application each.
// d_base != nullptr: the family starts from that device-resident one-stream state instead of the seed.
int init_mt19937(prand_state *st, uint64_t seed, Dist L, cudaStream_t stream, const void *d_base = nullptr)
{
    const unsigned lev_all = bit_length(st->first + st->ns - 1);
    const unsigned lev_tree = bit_length(st->ns - 1);
    std::vector<unsigned char> base;
    int rc = d_base ? PRAND_OK : build_seed_state(PRAND_MT19937, seed, base);
    if (rc) return rc;
    std::vector<host::MtPoly> polys;
    host::mt19937_levels(L, lev_all, polys);
    std::vector<MtOp> ops(lev_tree + 1);
    for (unsigned j = 0; j < lev_tree; j++) host::mt19937_to_op(polys[j], ops[j]);
    bool have_first = false;
    if (st->first) {                                   // x^(first L) = product of the levels of first's bits
        host::MtPoly acc;
        for (unsigned j = 0; j < lev_all; j++) {
            if (!((st->first >> j) & 1)) continue;
            if (!have_first) { acc = polys[j]; have_first = true; }
            else host::mt19937_mulmod(acc, acc, polys[j]);
        }
        host::mt19937_to_op(acc, ops[lev_tree]);
    }
    rc = ensure_ops(st, ops.size() * sizeof(MtOp));
    if (rc) return rc;
    UPLOAD(st->d_ops, ops.data(), ops.size() * sizeof(MtOp), stream);
    uint32_t *d = (uint32_t *)st->d_state[st->cur];
    if (d_base) { CU(cudaMemcpyAsync(d, d_base, stream_bytes(PRAND_MT19937), cudaMemcpyDeviceToDevice, stream)); }
    else UPLOAD(d, base.data(), base.size(), stream);
    const MtOp *d_ops = (const MtOp *)st->d_ops;
    LaunchInfo li;
    if (have_first) {
        CU(mt19937_apply(stream, d, d, 0, 1, 0, d_ops + lev_tree, &ops[lev_tree], &li));
        note(st, li);
    }
    for (unsigned j = 0; j < lev_tree; j++) {
        uint64_t lo = 1ull << j;
        uint64_t count = st->ns - lo < lo ? st->ns - lo : lo;
        CU(mt19937_apply(stream, d, d, lo, count, lo, d_ops + j, &ops[j], &li));
        note(st, li);
    }
    return PRAND_OK;
}

int init_body(prand_state *st, uint64_t seed, Dist L, cudaStream_t stream, const void *d_base = nullptr)
{
    if (st->gen == PRAND_MT19937) return init_mt19937(st, seed, L, stream, d_base);
    std::vector<unsigned char> base, ops;
    int rc = d_base ? PRAND_OK : build_seed_state(st->gen, seed, base);
    if (rc) return rc;
    if (d_base) base.assign(stream_bytes(st->gen), 0);
    const unsigned levels = bit_length(st->first + st->ns - 1);
    rc = build_level_ops(st->gen, L, levels, ops);
    if (rc) return rc;
    const size_t ops_off = (base.size() + 255) & ~(size_t)255;
    rc = ensure_ops(st, ops_off + ops.size() + 256);
    if (rc) return rc;
    if (d_base) { CU(cudaMemcpyAsync(st->d_ops, d_base, base.size(), cudaMemcpyDeviceToDevice, stream)); }
    else UPLOAD(st->d_ops, base.data(), base.size(), stream);
    if (!ops.empty())
        UPLOAD((char *)st->d_ops + ops_off, ops.data(), ops.size(), stream);
    JumpArgs a;
    a.base = st->d_ops;
    a.st_in = nullptr;
    a.st_out = st->d_state[st->cur];
    a.n_streams = st->ns;
    a.ops = (char *)st->d_ops + ops_off;
    a.idx0 = st->first;
    a.idx_stride = 1;
    a.count = 0;
    // GM/GQ with many streams: the paper's own relation (eq. 2-3) fills the family.
    // Streams 0 and 1 come from the jump kernel; then, level by level, stream s = k_n stream(s - 2^j)
    // - q_n stream(s - 2^(j+1)) with n = 2^j L -- two modular products per state word instead of one
    // matrix product per set bit of s.  the hook PRAND_GM_INIT=matrix keeps the matrix path.
    const bool tree = is_gm(st->gen) && st->ns >= 64 && !debug_hooks().gm_init_matrix;
    LaunchInfo li;
    if (!tree) {
        CU(launch_jump(stream, st->gen, a, &li, &L));
        note(st, li);
        return PRAND_OK;
    }
    a.count = 2;
    CU(launch_jump(stream, st->gen, a, &li));
    note(st, li);
    std::vector<uint64_t> kn, qn;
    const unsigned tlev = bit_length(st->ns - 1);
    host::gm_kq_levels(*gm_params(st->gen), L, tlev, kn, qn);
    for (unsigned j = 0; j < tlev; j++) {
        const uint64_t back = 1ull << j;
        for (int half = 0; half < 2; half++) {              // [2 back, 3 back) first: [3 back, 4 back) reads it
            const uint64_t lo = (2 + half) * back, hi = (3 + half) * back;
            if (lo >= st->ns) break;
            CU(gm_tree_fill(stream, st->gen, st->d_state[st->cur], st->ns, lo, hi < st->ns ? hi : st->ns, back,
                            kn[j], qn[j], &li));
            note(st, li);
        }
    }
    return PRAND_OK;
}

void destroy(prand_state *st)
{
    if (!st) return;
    // stream-ordered release: everything this state launched was on last_stream (the *_host calls
    // drain their copy stream before returning), so no device-wide synchronisation is needed
    cudaStream_t s = st->last_stream;
    for (int i = 0; i < 2; i++) {
        if (st->d_state[i]) cudaFreeAsync(st->d_state[i], s);
        if (st->d_stage[i]) cudaFreeAsync(st->d_stage[i], s);
        if (st->host_ready) { cudaEventDestroy(st->ev_gen[i]); cudaEventDestroy(st->ev_copy[i]); }
    }
    if (st->host_ready) cudaStreamDestroy(st->copy_stream);
    if (st->d_ops) cudaFreeAsync(st->d_ops, s);
    if (st->d_chunk_ops) cudaFreeAsync(st->d_chunk_ops, s);
    if (st->d_user_ops) cudaFreeAsync(st->d_user_ops, s);
    if (st->sec) { st->sec->last_stream = s; destroy(st->sec); }
    delete st;
}

}  // namespace

extern "C" int prand_init_shard(prand_state **out, int gen, uint64_t seed, uint64_t first_stream,
                                uint64_t n_streams, uint64_t block_len_mant, unsigned block_len_log2,
                                void *cuda_stream)
{
    if (!out) return PRAND_ERR_ARG;
    *out = nullptr;
    if (gen < 0 || gen >= PRAND_NGEN) return PRAND_ERR_GEN;
    if (n_streams == 0) return PRAND_ERR_ARG;
    if (block_len_mant == 0 && block_len_log2 != 0) return PRAND_ERR_ARG;
    if (block_len_log2 > 4096) return PRAND_ERR_ARG;
    if (first_stream + n_streams < first_stream) return PRAND_ERR_OVERFLOW;
    if (gen == PRAND_MT19937 && n_streams > PRAND_MT19937_MAX_STREAMS) return PRAND_ERR_ARG;
    if (gen == PRAND_MT19937 && !host::mt19937_phi_selfcheck()) return PRAND_ERR_INTERNAL;
    {
        unsigned __int128 top = (unsigned __int128)(first_stream + n_streams - 1) * block_len_mant;
        if (top >> 64) return PRAND_ERR_OVERFLOW;
    }
    {   // seed validity before any allocation
        std::vector<unsigned char> tmp;
        int rc = build_seed_state(gen, seed, tmp);
        if (rc) return rc;
    }
    prand_state *st = new (std::nothrow) prand_state();
    if (!st) return PRAND_ERR_ALLOC;
    std::memset(st, 0, sizeof *st);
    st->gm_clean = true;
    st->gen = gen;
    st->ns = n_streams;
    st->first = first_stream;
    st->bytes = (size_t)n_streams * stream_bytes(gen);
    st->last_kernel = "";
    st->last_stream = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaGetDevice(&st->device);
    if (e == cudaSuccess) e = dev_alloc(&st->d_state[0], st->bytes, st->last_stream);
    if (e != cudaSuccess) {
        delete st;
        g_last_cuda_error = (int)e;
        return e == cudaErrorMemoryAllocation ? PRAND_ERR_ALLOC : PRAND_ERR_CUDA;
    }
    Dist L = {block_len_mant, block_len_log2};
    int rc = init_body(st, seed, L, (cudaStream_t)cuda_stream);
    if (rc) { destroy(st); return rc; }
    *out = st;
    return PRAND_OK;
}

extern "C" int prand_init(prand_state **out, int gen, uint64_t seed, uint64_t n_streams,
                          uint64_t block_len_mant, unsigned block_len_log2, void *cuda_stream)
{
    return prand_init_shard(out, gen, seed, 0, n_streams, block_len_mant, block_len_log2, cuda_stream);
}

// ==================================================================================================
// prand_jump (a2)
// ==================================================================================================
namespace {
// upload the operator of distance n into st->d_ops
int jump_prepare(prand_state *st, Dist n, cudaStream_t stream)
{
    std::vector<unsigned char> ops;
    int rc = build_level_ops(st->gen, n, 1, ops);
    if (rc) return rc;
    rc = ensure_ops(st, ops.size());
    if (rc) return rc;
    UPLOAD(st->d_ops, ops.data(), ops.size(), stream);
    return PRAND_OK;
}
// apply the operator in st->d_ops to every stream
int jump_launch(prand_state *st, cudaStream_t stream, const Dist *dist = nullptr)
{
    LaunchInfo li;
    if (st->gen == PRAND_MT19937) {
        uint32_t *d = (uint32_t *)st->d_state[st->cur];
        CU(mt19937_apply(stream, d, d, 0, st->ns, 0, (const MtOp *)st->d_ops, nullptr, &li));
    } else {
        JumpArgs a;
        a.base = nullptr;
        a.st_in = st->d_state[st->cur];
        a.st_out = st->d_state[st->cur];     // one thread reads and writes its own words only
        a.n_streams = st->ns;
        a.ops = st->d_ops;
        a.idx0 = 1;                          // every stream applies level 0 exactly once
        a.idx_stride = 0;
        a.count = 0;
        CU(launch_jump(stream, st->gen, a, &li, dist));
    }
    note(st, li);
    return PRAND_OK;
}
}  // namespace

extern "C" int prand_jump(prand_state *st, uint64_t steps_mant, unsigned steps_log2, void *cuda_stream)
{
    if (!st) return PRAND_ERR_ARG;
    if (steps_log2 > 32768) return PRAND_ERR_ARG;
    if (steps_mant == 0) return PRAND_OK;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    st->last_stream = stream;
    Dist n = {steps_mant, steps_log2};
    if (st->gen == PRAND_MT19937) {
        // a tabulated distance is one application of a device-resident polynomial; any other
        // distance "reduces to jumping ahead blocks of lengths 2^i1, ..., 2^il" of the binary notation, applied
        // one after the other on the device -- no host polynomial arithmetic.  With many streams and many set
        // bits the applications cost more than the host products that merge them (~1.5 ms each against ~1 us
        // per stream and application): then the host multiplies the tabulated polynomials and one application runs.
        std::vector<int> terms;
        if (host::mt19937_table() && host::mt19937_table_terms(n, terms)) {
            const double app_us = st->ns < 100 ? 90.0 : 0.9 * (double)st->ns;
            const double device_us = terms.size() * app_us, host_us = (terms.size() - 1) * 1500.0 + app_us;
            if (const MtOp *table = device_us <= host_us ? mt_device_table(stream) : nullptr) {
                uint32_t *d = (uint32_t *)st->d_state[st->cur];
                for (int t : terms) {
                    LaunchInfo li;
                    CU(mt19937_apply(stream, d, d, 0, st->ns, 0, table + t, (const MtOp *)host::mt19937_table() + t, &li));
                    li.kernel = "mt19937_apply<table>";
                    note(st, li);
                }
                return PRAND_OK;
            }
        }
    }
    int rc = jump_prepare(st, n, stream);
    if (rc) return rc;
    rc = jump_launch(st, stream, &n);
    if (rc) return rc;
    if (steps_log2 >= 4 || steps_mant >= 16) st->gm_clean = true;   // past the 2-adic transient
    return PRAND_OK;
}

// ==================================================================================================
// prand_generate_* (a3-a8)
// ==================================================================================================
namespace {

// Launch policy.  With few streams one thread per stream (group) leaves the GPU idle,
// so a stream's range is cut into sub-sections reached by jump-ahead; outputs are
// defined by position, so this changes nothing but the schedule.  MT19937 never chunks: applying its
// jump polynomial costs as much as generating ~10^5 outputs; its kernel is CTA-cooperative instead.
void plan_chunks(int gen, uint64_t ns, uint64_t n, int dtype, int sms, uint64_t *chunk_len, uint64_t *n_chunks)
{
    *chunk_len = n;
    *n_chunks = 1;
    if (gen == PRAND_MT19937 || n == 0) return;
    const uint64_t forced = debug_hooks().chunk_len;
    uint64_t len;
    if (forced) {
        len = forced;
    } else {
        // threads one launch gets without chunking
        uint64_t per_thread_streams = 1, lanes_per_stream = 1, min_len = 64;
        if (gen == PRAND_LFSR113) per_thread_streams = lfsr113_narrow(ns, n, dtype, sms) ? 1 : 4;
        else if (gen == PRAND_MRG32K3A) per_thread_streams = dtype == DT_F64 ? 2 : 4;
        else {
            min_len = 128;
            if (gen == PRAND_GM61) lanes_per_stream = 4;
        }
        uint64_t threads = ns * lanes_per_stream / per_thread_streams;
        if (threads == 0) threads = 1;
        // one balanced wave: as many equal chunks as fit the threads resident at once, never more
        // (a second, partial wave would cost a whole chunk time)
        const uint64_t capacity = (uint64_t)sms * 1024;
        // the store-bound kernels (LFSR113, MRG32K3A with 8-byte outputs) are the exception: measured on B200, sub-sections
        // of about 1024 rows in several waves beat one wave of long ones (C2: 4 x 4096 rows 1.379 ms, 16 x 1024 rows
        // 1.294 ms; C5-lfsr113: unchunked 1.341 ms, 2 x 1024 rows 1.301 ms) -- CTAs are handed out in index order, so the
        // rows being written at any moment stay close together in DRAM, and a retiring CTA is replaced at once; below
        // ~512 rows the jump to a sub-section's start costs more than that gains
        const bool store_bound = gen == PRAND_LFSR113 || (gen == PRAND_MRG32K3A && dtype == DT_F64);
        const uint64_t wave_len = 1024;
        if (2 * threads > capacity) {
            if (!store_bound || n < 2 * wave_len) return;
            len = wave_len;
        } else {
            const uint64_t want = capacity / threads;
            len = (n + want - 1) / want;
            if (len < min_len) len = min_len;
            if (store_bound && len > wave_len) len = wave_len;
        }
    }
    // whole row blocks per chunk: 32 for LFSR113's bit-stream form, else 12 (4: row groups of the
    // 4-lane GM path; 3: MRG32K3A's renamed rotation)
    const uint64_t gran = gen == PRAND_LFSR113 ? 32 : 12;
    len = (len + gran - 1) / gran * gran;
    if (len >= n) return;
    if ((n + len - 1) / len > 65535) len = ((n + 65534) / 65535 + gran - 1) / gran * gran;   // chunks ride on gridDim.y
    *chunk_len = len;
    *n_chunks = (n + len - 1) / len;
}

int ensure_chunk_ops(prand_state *st, uint64_t chunk_len, uint64_t n_chunks, cudaStream_t stream)
{
    if (st->d_chunk_ops && st->chunk_len == chunk_len && st->chunk_count >= n_chunks) return PRAND_OK;
    // operator of distance c * chunk_len for c = 1..n_chunks-1: one application per virtual stream.  The host
    // bytes of the most recent (generator, chunk_len, n_chunks) plans are kept for the process, so that a state
    // created per step (init + generate + free) does not pay the preparation again.
    struct Plan { int gen; uint64_t len, n; std::vector<unsigned char> bytes; };
    static std::mutex mu;
    static std::vector<Plan> plans;                        // most recent last, at most 8
    std::vector<unsigned char> ops;
    {
        std::lock_guard<std::mutex> lock(mu);
        for (const Plan &p : plans)
            if (p.gen == st->gen && p.len == chunk_len && p.n == n_chunks) ops = p.bytes;
    }
    if (ops.empty()) {
        std::vector<unsigned char> one;
        for (uint64_t c = 1; c < n_chunks; c++) {
            Dist d = {c * chunk_len, 0};
            int rc = build_level_ops(st->gen, d, 1, one);
            if (rc) return rc;
            ops.insert(ops.end(), one.begin(), one.end());
        }
        std::lock_guard<std::mutex> lock(mu);
        if (plans.size() == 8) plans.erase(plans.begin());
        plans.push_back(Plan{st->gen, chunk_len, n_chunks, ops});
    }
    if (st->d_chunk_ops) { CU(cudaFreeAsync(st->d_chunk_ops, stream)); st->d_chunk_ops = nullptr; }
    CU(dev_alloc(&st->d_chunk_ops, ops.size(), stream));
    UPLOAD(st->d_chunk_ops, ops.data(), ops.size(), stream);
    st->chunk_len = chunk_len;
    st->chunk_count = n_chunks;
    return PRAND_OK;
}

// peek: the numbers are produced but the streams do not advance (the advanced state goes to the spare buffer and is
// dropped) -- what the skip-per-step generator needs before it jumps
int generate(prand_state *st, void *out, uint64_t n, int dtype, cudaStream_t stream, bool peek = false)
{
    if (!st || (!out && n)) return PRAND_ERR_ARG;
    if (n == 0) return PRAND_OK;
    st->last_stream = stream;
    const size_t esz = dtype == DT_F64 ? 8 : 4;
    if ((uintptr_t)out % esz) return PRAND_ERR_ARG;
    {
        unsigned __int128 total = (unsigned __int128)n * st->ns * esz;
        if (total >> 62) return PRAND_ERR_OVERFLOW;
    }
    GenArgs a;
    a.out = out;
    a.dtype = dtype;
    a.n_streams = st->ns;
    a.n = n;
    plan_chunks(st->gen, st->ns, n, dtype, sm_count(), &a.chunk_len, &a.n_chunks);
    a.chunk_ops = nullptr;
    a.clean = st->gm_clean;
    a.st_in = st->d_state[st->cur];
    a.st_out = st->d_state[st->cur];
    if (a.n_chunks > 1 || peek) {
        // chunk c reads the start state while the last chunk writes the final one: separate buffers
        int rc = ensure_second_buffer(st);
        if (rc) return rc;
        if (a.n_chunks > 1) {
            rc = ensure_chunk_ops(st, a.chunk_len, a.n_chunks, stream);
            if (rc) return rc;
            a.chunk_ops = st->d_chunk_ops;
        }
        a.st_out = st->d_state[1 - st->cur];
    }
    LaunchInfo li = {"", 0};
    cudaError_t e;
    if (st->gen == PRAND_LFSR113) e = lfsr113_generate(stream, a, &li);
    else if (st->gen == PRAND_MRG32K3A) e = mrg32k3a_generate(stream, a, &li);
    else if (st->gen == PRAND_MT19937) e = mt19937_generate(stream, a, &li);
    else e = gm_generate(stream, st->gen, a, &li);
    if (e != cudaSuccess) return cuda_fail(e);
    note(st, li);
    if (peek) return PRAND_OK;
    if (a.n_chunks > 1) st->cur = 1 - st->cur;
    if (n >= 16) st->gm_clean = true;
    return PRAND_OK;
}

// rng_generate_array_: generate on the device in row blocks, copy each block back
// while the next one is generated.
int ensure_host_path(prand_state *st, size_t want_bytes)
{
    if (!st->host_ready) {
        CU(cudaStreamCreateWithFlags(&st->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; i++) {
            CU(cudaEventCreateWithFlags(&st->ev_gen[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&st->ev_copy[i], cudaEventDisableTiming));
        }
        st->host_ready = true;
    }
    if (st->stage_bytes < want_bytes) {
        for (int i = 0; i < 2; i++) {      // earlier *_host calls drained both streams before returning
            if (st->d_stage[i]) { CU(cudaFreeAsync(st->d_stage[i], st->last_stream)); st->d_stage[i] = nullptr; }
            CU(dev_alloc(&st->d_stage[i], want_bytes, st->last_stream));
        }
        st->stage_bytes = want_bytes;
    }
    return PRAND_OK;
}

int generate_host(prand_state *st, void *host_out, uint64_t n, int dtype, cudaStream_t stream)
{
    if (!st || (!host_out && n)) return PRAND_ERR_ARG;
    if (n == 0) return PRAND_OK;
    st->last_stream = stream;
    const size_t esz = dtype == DT_F64 ? 8 : 4;
    const size_t row_bytes = (size_t)st->ns * esz;
    const size_t block_target = (size_t)256 << 20;
    uint64_t rows_per_block = block_target / row_bytes;
    if (rows_per_block == 0) rows_per_block = 1;
    if (rows_per_block > n) rows_per_block = n;
    int rc = ensure_host_path(st, rows_per_block * row_bytes);
    if (rc) return rc;
    int slot = 0;
    uint64_t blocks = 0;
    for (uint64_t r0 = 0; r0 < n; r0 += rows_per_block, slot ^= 1, blocks++) {
        const uint64_t rows = n - r0 < rows_per_block ? n - r0 : rows_per_block;
        if (blocks >= 2) CU(cudaStreamWaitEvent(stream, st->ev_copy[slot], 0));   // slot's previous copy done
        rc = generate(st, st->d_stage[slot], rows, dtype, stream);
        if (rc) return rc;
        CU(cudaEventRecord(st->ev_gen[slot], stream));
        CU(cudaStreamWaitEvent(st->copy_stream, st->ev_gen[slot], 0));
        CU(cudaMemcpyAsync((char *)host_out + r0 * row_bytes, st->d_stage[slot], rows * row_bytes,
                           cudaMemcpyDeviceToHost, st->copy_stream));
        CU(cudaEventRecord(st->ev_copy[slot], st->copy_stream));
    }
    CU(cudaStreamSynchronize(st->copy_stream));
    CU(cudaStreamSynchronize(stream));
    return PRAND_OK;
}

}  // namespace

extern "C" int prand_generate_u32(prand_state *st, uint32_t *out, uint64_t n, void *s)
{
    return generate(st, out, n, DT_U32, (cudaStream_t)s);
}
extern "C" int prand_generate_f32(prand_state *st, float *out, uint64_t n, void *s)
{
    return generate(st, out, n, DT_F32, (cudaStream_t)s);
}
extern "C" int prand_generate_f64(prand_state *st, double *out, uint64_t n, void *s)
{
    return generate(st, out, n, DT_F64, (cudaStream_t)s);
}
extern "C" int prand_generate_u32_host(prand_state *st, uint32_t *out, uint64_t n, void *s)
{
    return generate_host(st, out, n, DT_U32, (cudaStream_t)s);
}
extern "C" int prand_generate_f32_host(prand_state *st, float *out, uint64_t n, void *s)
{
    return generate_host(st, out, n, DT_F32, (cudaStream_t)s);
}
extern "C" int prand_generate_f64_host(prand_state *st, double *out, uint64_t n, void *s)
{
    return generate_host(st, out, n, DT_F64, (cudaStream_t)s);
}

namespace prand {
int record_cuda_error(cudaError_t e) { return cuda_fail(e); }
void count_launches(unsigned n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
}  // namespace prand

// ==================================================================================================
// prand_generate_seq_* (SURVEY.md 8(f)1): PRAND's single-sequence array fill
// ==================================================================================================
namespace {

// PAPER.md:382, Table 5: the array is divided into sections, each section is
// reached by jump-ahead and filled in parallel; the result is what the serial generator would have
// produced.  Here: section c = a stream that starts c * sec_len ahead of the state, the family is
// filled in the interleaved layout by the bulk kernels and transposed into out[c * sec_len + i].
void plan_sections(int gen, uint64_t length, uint64_t *n_sections, uint64_t *sec_len, int sms = 148)
{
    // enough sections to fill the GPU, sections long enough to amortise the jump to their start
    const uint64_t min_len = gen == PRAND_MT19937 ? 8 * 624 : 1024;
    // MT19937: every section costs a polynomial application (~1 us of a whole SM): one CTA of four sections per SM
    // others: one section per thread; 2^17 sections are one wave of 28 warps per SM on 148 SMs
    uint64_t max_sec = gen == PRAND_MT19937 ? 4 * (uint64_t)sms : 131072;
    if (gen != PRAND_MT19937 && debug_hooks().seq_sections) max_sec = debug_hooks().seq_sections;   // tuning hook
    uint64_t S = length / min_len;
    if (S > max_sec) S = max_sec;
    if (S < 1) S = 1;
    uint64_t L = (length + S - 1) / S;
    L = (L + 31) / 32 * 32;
    *sec_len = L;
    *n_sections = (length + L - 1) / L;
}

int generate_seq(prand_state *st, void *out, uint64_t length, int dtype, cudaStream_t stream)
{
    if (!st || (!out && length)) return PRAND_ERR_ARG;
    if (st->ns != 1) return PRAND_ERR_ARG;                 // one sequence: the state of a single stream
    if (length == 0) return PRAND_OK;
    uint64_t S, L;
    plan_sections(st->gen, length, &S, &L, sm_count());
    if (S == 1) return generate(st, out, length, dtype, stream);
    st->last_stream = stream;
    const size_t esz = dtype == DT_F64 ? 8 : 4;
    if ((uintptr_t)out % esz) return PRAND_ERR_ARG;
    // the family of sections (cached across calls of the same shape)
    if (st->sec && st->sec->ns != S) { st->sec->last_stream = stream; destroy(st->sec); st->sec = nullptr; }
    if (!st->sec) {
        prand_state *c = new (std::nothrow) prand_state();
        if (!c) return PRAND_ERR_ALLOC;
        std::memset(c, 0, sizeof *c);
        c->gen = st->gen;
        c->ns = S;
        c->bytes = (size_t)S * stream_bytes(st->gen);
        c->last_kernel = "";
        c->last_stream = stream;
        c->device = st->device;
        cudaError_t e = dev_alloc(&c->d_state[0], c->bytes, stream);
        if (e != cudaSuccess) { delete c; return cuda_fail(e); }
        st->sec = c;
    }
    prand_state *c = st->sec;
    c->cur = 0;
    c->gm_clean = st->gm_clean;
    c->last_stream = stream;
    Dist Ld = {L, 0};
    int rc = init_body(c, 0, Ld, stream, st->d_state[st->cur]);
    if (rc) return rc;
    if (st->gen == PRAND_MRG32K3A && dtype == DT_F64 && (uintptr_t)out % 16 == 0) {
        // fused path: the sections are written in place, no scratch buffer, no transposition
        LaunchInfo li;
        CU(mrg32k3a_seq_f64(stream, c->d_state[c->cur], st->d_state[st->cur], (double *)out, S, L, length, &li));
        note(st, li);
        return PRAND_OK;                                       // the kernel left the advanced state in st
    }
    if (st->gen == PRAND_MT19937 && (uintptr_t)out % 16 == 0) {
        // per-stream thread groups write each section's numbers as contiguous runs straight from registers
        LaunchInfo li;
        CU(mt19937_seq(stream, c->d_state[c->cur], st->d_state[st->cur], out, dtype, S, L, length, &li));
        note(st, li);
        return PRAND_OK;
    }
    if (st->gen == PRAND_MRG32K3A && dtype != DT_F64 && (uintptr_t)out % 16 == 0) {
        LaunchInfo li;
        CU(mrg32k3a_seq4(stream, c->d_state[c->cur], out, dtype, S, L, length, &li));
        note(st, li);
        return prand_jump(st, length, 0, stream);          // the sequence has advanced by `length`
    }
    if (st->gen == PRAND_LFSR113 && (uintptr_t)out % 16 == 0) {
        // one section per thread, 32-row blocks transposed through a per-warp shared-memory tile
        LaunchInfo li;
        CU(lfsr113_seq(stream, c->d_state[c->cur], out, dtype, S, L, length, &li));
        note(st, li);
        return prand_jump(st, length, 0, stream);          // the sequence has advanced by `length`
    }
    void *tmp = nullptr;
    CU(dev_alloc(&tmp, (size_t)L * S * esz, stream));
    rc = generate(c, tmp, L, dtype, stream);
    if (rc == PRAND_OK) {
        LaunchInfo li;
        cudaError_t e = transpose_sections(stream, tmp, out, S, L, length, (int)esz, &li);
        if (e != cudaSuccess) rc = cuda_fail(e);
        else note(st, li);
        st->last_kernel = c->last_kernel;
    }
    CU(cudaFreeAsync(tmp, stream));
    if (rc) return rc;
    return prand_jump(st, length, 0, stream);              // the sequence has advanced by `length`
}

}  // namespace

// prand_generate_strided_* (SURVEY.md 8(f)4): the sequence that skips ahead after every output
// (Table 3 PAPER.md:249-275 tests such sequences for skips of 2^n).  Row i holds every
// stream's output at position P + i * stride: the output is produced from a copy of the state, the
// state itself jumps by `stride` with one prepared operator: two launches per row, no copy of the state.
namespace {
int generate_strided(prand_state *st, void *out, uint64_t n, int dtype, Dist stride, cudaStream_t stream)
{
    if (!st || (!out && n)) return PRAND_ERR_ARG;
    if (stride.mant == 0 || stride.log2 > 32768) return PRAND_ERR_ARG;
    if (n == 0) return PRAND_OK;
    if (stride.mant == 1 && stride.log2 == 0) return generate(st, out, n, dtype, stream);
    st->last_stream = stream;
    const size_t esz = dtype == DT_F64 ? 8 : 4;
    if ((uintptr_t)out % esz) return PRAND_ERR_ARG;
    int rc = ensure_second_buffer(st);
    if (rc) return rc;
    rc = jump_prepare(st, stride, stream);
    if (rc) return rc;
    const bool clean0 = st->gm_clean;
    for (uint64_t i = 0; i < n; i++) {
        // one output per stream without advancing it (the stepped state lands in the spare buffer: no state copy)
        rc = generate(st, (char *)out + i * st->ns * esz, 1, dtype, stream, true);
        if (rc) return rc;
        rc = jump_launch(st, stream);
        if (rc) return rc;
        if (stride.log2 >= 4 || stride.mant >= 16) st->gm_clean = true;
        else st->gm_clean = clean0 && st->gm_clean;
    }
    return PRAND_OK;
}
}  // namespace

extern "C" int prand_generate_strided_u32(prand_state *st, uint32_t *out, uint64_t n, uint64_t stride_mant,
                                          unsigned stride_log2, void *s)
{
    return generate_strided(st, out, n, DT_U32, Dist{stride_mant, stride_log2}, (cudaStream_t)s);
}
extern "C" int prand_generate_strided_f32(prand_state *st, float *out, uint64_t n, uint64_t stride_mant,
                                          unsigned stride_log2, void *s)
{
    return generate_strided(st, out, n, DT_F32, Dist{stride_mant, stride_log2}, (cudaStream_t)s);
}
extern "C" int prand_generate_strided_f64(prand_state *st, double *out, uint64_t n, uint64_t stride_mant,
                                          unsigned stride_log2, void *s)
{
    return generate_strided(st, out, n, DT_F64, Dist{stride_mant, stride_log2}, (cudaStream_t)s);
}

extern "C" int prand_generate_seq_u32(prand_state *st, uint32_t *out, uint64_t length, void *s)
{
    return generate_seq(st, out, length, DT_U32, (cudaStream_t)s);
}
extern "C" int prand_generate_seq_f32(prand_state *st, float *out, uint64_t length, void *s)
{
    return generate_seq(st, out, length, DT_F32, (cudaStream_t)s);
}
extern "C" int prand_generate_seq_f64(prand_state *st, double *out, uint64_t length, void *s)
{
    return generate_seq(st, out, length, DT_F64, (cudaStream_t)s);
}

// ==================================================================================================
// device-callable API support
// ==================================================================================================
extern "C" void *prand_state_device_ptr(prand_state *st)
{
    return st ? st->d_state[st->cur] : nullptr;
}
extern "C" uint64_t prand_state_n_streams(const prand_state *st) { return st ? st->ns : 0; }

extern "C" int prand_device_ops(prand_state *st, uint64_t dist_mant, unsigned dist_log2, unsigned levels,
                                const void **d_ops, void *cuda_stream)
{
    if (!st || !d_ops || levels == 0 || levels > 64 || dist_log2 > 32768) return PRAND_ERR_ARG;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    st->last_stream = stream;
    std::vector<unsigned char> ops;
    int rc = build_level_ops(st->gen, Dist{dist_mant, dist_log2}, levels, ops);
    if (rc) return rc;
    if (st->d_user_ops) { CU(cudaFreeAsync(st->d_user_ops, stream)); st->d_user_ops = nullptr; }
    CU(dev_alloc(&st->d_user_ops, ops.size(), stream));
    UPLOAD(st->d_user_ops, ops.data(), ops.size(), stream);
    CU(cudaStreamSynchronize(stream));                 // the host vector goes out of scope
    *d_ops = st->d_user_ops;
    return PRAND_OK;
}

namespace {
int devapi_init_fill(prand_state *st, uint64_t mant, unsigned log2, uint64_t ns, void *out, uint64_t n, int dtype,
                     cudaStream_t stream)
{
    if (!st || (!out && n) || ns == 0) return PRAND_ERR_ARG;
    if (st->ns != 1) return PRAND_ERR_ARG;                 // the base stream
    {
        unsigned __int128 top = (unsigned __int128)(ns - 1) * mant;
        if (top >> 64) return PRAND_ERR_OVERFLOW;
    }
    const void *ops = nullptr;
    const unsigned levels = ns > 1 ? bit_length(ns - 1) : 1;
    int rc = prand_device_ops(st, mant, log2, levels, &ops, stream);
    if (rc) return rc;
    if (n == 0) return PRAND_OK;
    LaunchInfo li = {"", 0};
    cudaError_t e = devapi_init_generate(stream, st->gen, st->d_state[st->cur], ops, out, ns, n, dtype, &li);
    if (e != cudaSuccess) return cuda_fail(e);
    note(st, li);
    return PRAND_OK;
}
}  // namespace
extern "C" int prand_device_api_init_fill_u32(prand_state *st, uint64_t m, unsigned l, uint64_t ns, uint32_t *out, uint64_t n, void *s)
{
    return devapi_init_fill(st, m, l, ns, out, n, DT_U32, (cudaStream_t)s);
}
extern "C" int prand_device_api_init_fill_f32(prand_state *st, uint64_t m, unsigned l, uint64_t ns, float *out, uint64_t n, void *s)
{
    return devapi_init_fill(st, m, l, ns, out, n, DT_F32, (cudaStream_t)s);
}
extern "C" int prand_device_api_init_fill_f64(prand_state *st, uint64_t m, unsigned l, uint64_t ns, double *out, uint64_t n, void *s)
{
    return devapi_init_fill(st, m, l, ns, out, n, DT_F64, (cudaStream_t)s);
}

namespace {
int devapi_fill(prand_state *st, void *out, uint64_t n, int dtype, cudaStream_t stream)
{
    if (!st || (!out && n)) return PRAND_ERR_ARG;
    if (n == 0) return PRAND_OK;
    st->last_stream = stream;
    LaunchInfo li = {"", 0};
    cudaError_t e = devapi_generate(stream, st->gen, st->d_state[st->cur], out, st->ns, n, dtype, &li);
    if (e != cudaSuccess) return cuda_fail(e);
    note(st, li);
    if (n >= 16) st->gm_clean = true;
    return PRAND_OK;
}
}  // namespace
extern "C" int prand_device_api_fill_u32(prand_state *st, uint32_t *out, uint64_t n, void *s)
{
    return devapi_fill(st, out, n, DT_U32, (cudaStream_t)s);
}
extern "C" int prand_device_api_fill_f32(prand_state *st, float *out, uint64_t n, void *s)
{
    return devapi_fill(st, out, n, DT_F32, (cudaStream_t)s);
}
extern "C" int prand_device_api_fill_f64(prand_state *st, double *out, uint64_t n, void *s)
{
    return devapi_fill(st, out, n, DT_F64, (cudaStream_t)s);
}

// ==================================================================================================
// canonical state export / import
// ==================================================================================================
namespace {

// internal word (w, s) lives at index w * ns + s (SoA) except MT19937, which is [s][624] already
template <class W> void soa_to_canon(const W *soa, W *canon, uint64_t ns, size_t words)
{
    for (size_t w = 0; w < words; w++)
        for (uint64_t s = 0; s < ns; s++) canon[s * words + w] = soa[w * ns + s];
}
template <class W> void canon_to_soa(const W *canon, W *soa, uint64_t ns, size_t words)
{
    for (size_t w = 0; w < words; w++)
        for (uint64_t s = 0; s < ns; s++) soa[w * ns + s] = canon[s * words + w];
}

}  // namespace

extern "C" size_t prand_state_bytes(const prand_state *st) { return st ? st->bytes : 0; }
extern "C" uint64_t prand_n_streams(const prand_state *st) { return st ? st->ns : 0; }
extern "C" int prand_gen_of(const prand_state *st) { return st ? st->gen : PRAND_ERR_ARG; }

extern "C" int prand_get_state(const prand_state *st, void *host_buf, size_t bytes)
{
    if (!st || !host_buf) return PRAND_ERR_ARG;
    if (bytes != st->bytes) return PRAND_ERR_SIZE;
    CU(cudaDeviceSynchronize());
    const size_t words = state_words(st->gen);
    if (st->gen == PRAND_MT19937) {
        CU(cudaMemcpy(host_buf, st->d_state[st->cur], bytes, cudaMemcpyDeviceToHost));
        uint32_t *w = (uint32_t *)host_buf;
        for (uint64_t s = 0; s < st->ns; s++) w[s * words] &= 0x80000000u;   // reading T2
        return PRAND_OK;
    }
    std::vector<unsigned char> tmp(bytes);
    CU(cudaMemcpy(tmp.data(), st->d_state[st->cur], bytes, cudaMemcpyDeviceToHost));
    if (state_word_bytes(st->gen) == 8) soa_to_canon((const uint64_t *)tmp.data(), (uint64_t *)host_buf, st->ns, words);
    else soa_to_canon((const uint32_t *)tmp.data(), (uint32_t *)host_buf, st->ns, words);
    if (st->gen == PRAND_LFSR113) {                 // reading L3: only the top p bits are state
        static const uint32_t mask[4] = {0xFFFFFFFEu, 0xFFFFFFF8u, 0xFFFFFFF0u, 0xFFFFFF80u};
        uint32_t *w = (uint32_t *)host_buf;
        for (uint64_t s = 0; s < st->ns; s++)
            for (int c = 0; c < 4; c++) w[4 * s + c] &= mask[c];
    }
    return PRAND_OK;
}

extern "C" int prand_set_state(prand_state *st, const void *host_buf, size_t bytes)
{
    if (!st || !host_buf) return PRAND_ERR_ARG;
    if (bytes != st->bytes) return PRAND_ERR_SIZE;
    CU(cudaDeviceSynchronize());
    const size_t words = state_words(st->gen);
    if (st->gen == PRAND_MT19937) {
        CU(cudaMemcpy(st->d_state[st->cur], host_buf, bytes, cudaMemcpyHostToDevice));
        return PRAND_OK;
    }
    // the kernels' exactness arguments assume canonical residues and live (non-degenerate) components
    if (st->gen == PRAND_LFSR113) {
        static const uint32_t top[4] = {0xFFFFFFFEu, 0xFFFFFFF8u, 0xFFFFFFF0u, 0xFFFFFF80u};
        const uint32_t *w = (const uint32_t *)host_buf;
        for (uint64_t i = 0; i < st->ns * 4; i++)
            if ((w[i] & top[i & 3]) == 0) return PRAND_ERR_ARG;                 // a component stuck at zero
    } else if (st->gen == PRAND_MRG32K3A) {
        const uint32_t *w = (const uint32_t *)host_buf;
        for (uint64_t s = 0; s < st->ns; s++, w += 6) {
            for (int k = 0; k < 6; k++)
                if (w[k] >= (k < 3 ? 4294967087u : 4294944443u)) return PRAND_ERR_ARG;   // not a residue mod m1 / m2
            if ((w[0] | w[1] | w[2]) == 0 || (w[3] | w[4] | w[5]) == 0) return PRAND_ERR_ARG;
        }
    } else if (const GmParams *gp = gm_params(st->gen)) {
        if (gp->wide) {
            const uint64_t *w = (const uint64_t *)host_buf;
            for (size_t i = 0; i < st->ns * words; i++)
                if (w[i] >= gp->g) return PRAND_ERR_ARG;
        } else {
            const uint32_t *w = (const uint32_t *)host_buf;
            for (size_t i = 0; i < st->ns * words; i++)
                if (w[i] >= gp->g) return PRAND_ERR_ARG;
        }
    }
    std::vector<unsigned char> tmp(bytes);
    if (const GmParams *gp = gm_params(st->gen)) {
        // GM55/GQ58 (g = 2^t p): the fast kernels need every word to be a multiple of 2^t
        st->gm_clean = true;
        const uint64_t odd_g = gp->g & (0 - gp->g);          // 2^t
        if (odd_g > 1 && gp->wide) {
            const uint64_t *w = (const uint64_t *)host_buf;
            for (size_t i = 0; i < st->ns * words && st->gm_clean; i++)
                if (w[i] & (odd_g - 1)) st->gm_clean = false;
        }
    }
    if (state_word_bytes(st->gen) == 8) canon_to_soa((const uint64_t *)host_buf, (uint64_t *)tmp.data(), st->ns, words);
    else canon_to_soa((const uint32_t *)host_buf, (uint32_t *)tmp.data(), st->ns, words);
    CU(cudaMemcpy(st->d_state[st->cur], tmp.data(), bytes, cudaMemcpyHostToDevice));
    return PRAND_OK;
}

extern "C" int prand_free(prand_state *st)
{
    if (!st) return PRAND_ERR_ARG;
    destroy(st);
    return PRAND_OK;
}

// ==================================================================================================
// probes and bookkeeping
// ==================================================================================================
extern "C" int prand_fill_u32(uint32_t *out, uint64_t n_words, uint32_t value, void *cuda_stream)
{
    if (!out && n_words) return PRAND_ERR_ARG;
    if ((uintptr_t)out % 16) return PRAND_ERR_ARG;
    if (n_words == 0) return PRAND_OK;
    LaunchInfo li = {"", 0};
    CU(fill_u32((cudaStream_t)cuda_stream, out, n_words, value, &li));
    note(nullptr, li);
    return PRAND_OK;
}

extern "C" int prand_trim(void)
{
    int dev = 0;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (dev >= 0 && dev < 64 && g_pools[dev]) CU(cudaMemPoolTrimTo(g_pools[dev], 0));
    return PRAND_OK;
}

extern "C" int prand_debug_set(const char *name, const char *value)
{
    if (!name) return PRAND_ERR_ARG;
    bool known = false;
    for (const char *n : HOOK_NAMES) known = known || std::string(n) == name;
    if (!known) return PRAND_ERR_ARG;
    debug_hooks();                                         // environment first, once
    std::lock_guard<std::mutex> lock(g_hooks_mu);
    hook_assign(g_hooks, name, value);
    return PRAND_OK;
}

extern "C" uint64_t prand_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
extern "C" uint64_t prand_uploaded_bytes(void) { return g_h2d_bytes.load(std::memory_order_relaxed); }
extern "C" const char *prand_last_kernel(const prand_state *st) { return st ? st->last_kernel : ""; }
extern "C" int prand_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" const char *prand_version(void) { return "prand-b200 0.1 (sm_100a)"; }

extern "C" const char *prand_strerror(int code)
{
    switch (code) {
    case PRAND_OK: return "ok";
    case PRAND_ERR_GEN: return "unknown generator";
    case PRAND_ERR_ARG: return "invalid argument";
    case PRAND_ERR_SEED: return "seed not valid for this generator";
    case PRAND_ERR_OVERFLOW: return "stream index times block length mantissa overflows 64 bits";
    case PRAND_ERR_CUDA: return "CUDA runtime error";
    case PRAND_ERR_SIZE: return "byte count does not match prand_state_bytes()";
    case PRAND_ERR_ALLOC: return "allocation failed";
    case PRAND_ERR_INTERNAL: return "internal self-check failed";
    case PRAND_ERR_CAPACITY: return "request exceeds the fixed capacity of the no-allocation entry point";
    default: return "unknown error code";
    }
}

// ==================================================================================================
// host-only hooks (include/prand_host.h)
// ==================================================================================================
extern "C" size_t prand_host_skip_op_bytes(int gen)
{
    if (gen == PRAND_LFSR113) return sizeof(LfsrOp);
    if (gen == PRAND_MRG32K3A) return sizeof(MrgOp);
    if (gen == PRAND_MT19937) return sizeof(MtOp);
    if (is_gm(gen)) return sizeof(GmOp);
    return 0;
}

extern "C" int prand_host_skip_op(int gen, uint64_t mant, unsigned log2, void *buf, size_t bytes)
{
    if (gen < 0 || gen >= PRAND_NGEN) return PRAND_ERR_GEN;
    if (!buf) return PRAND_ERR_ARG;
    if (bytes != prand_host_skip_op_bytes(gen)) return PRAND_ERR_SIZE;
    std::vector<unsigned char> ops;
    Dist n = {mant, log2};
    int rc = build_level_ops(gen, n, 1, ops);
    if (rc) return rc;
    std::memcpy(buf, ops.data(), bytes);
    return PRAND_OK;
}

extern "C" size_t prand_host_state_bytes(int gen) { return (gen < 0 || gen >= PRAND_NGEN) ? 0 : stream_bytes(gen); }

extern "C" int prand_host_seed_state(int gen, uint64_t seed, void *buf, size_t bytes)
{
    if (gen < 0 || gen >= PRAND_NGEN) return PRAND_ERR_GEN;
    if (!buf) return PRAND_ERR_ARG;
    if (bytes != stream_bytes(gen)) return PRAND_ERR_SIZE;
    std::vector<unsigned char> st;
    int rc = build_seed_state(gen, seed, st);
    if (rc) return rc;
    std::memcpy(buf, st.data(), bytes);
    return PRAND_OK;
}

extern "C" int prand_host_mt19937_phi(uint32_t *words624)
{
    if (!words624) return PRAND_ERR_ARG;
    MtOp op;
    host::mt19937_to_op(host::mt19937_phi(), op);
    std::memcpy(words624, op.w, sizeof op.w);
    return PRAND_OK;
}

extern "C" int prand_host_mt19937_phi_selfcheck(void)
{
    return host::mt19937_phi_selfcheck() ? PRAND_OK : PRAND_ERR_INTERNAL;
}

extern "C" int prand_host_mt19937_mulmod(const uint32_t *a624, const uint32_t *b624, uint32_t *r624)
{
    if (!a624 || !b624 || !r624) return PRAND_ERR_ARG;
    host::MtPoly a, b, r;
    std::memcpy(a.w, a624, sizeof a.w);            // little-endian: two u32 words per u64 word
    std::memcpy(b.w, b624, sizeof b.w);
    host::mt19937_mulmod(r, a, b);
    std::memcpy(r624, r.w, sizeof r.w);
    return PRAND_OK;
}

extern "C" int prand_host_mt19937_table(uint64_t mant, unsigned log2, uint32_t *words624)
{
    if (!words624 || log2 > 32768) return PRAND_ERR_ARG;
    const host::MtPoly *t = host::mt19937_table();
    const int idx = t ? host::mt19937_table_index(Dist{mant, log2}) : -1;
    if (idx < 0) return PRAND_ERR_ARG;
    std::memcpy(words624, t[idx].w, sizeof t[idx].w);
    return PRAND_OK;
}

extern "C" int prand_host_gm_kq(int gen, uint64_t mant, unsigned log2, uint64_t *k_n, uint64_t *q_n)
{
    const GmParams *p = gm_params(gen);
    if (!p) return PRAND_ERR_GEN;
    if (!k_n || !q_n || log2 > 32768) return PRAND_ERR_ARG;
    std::vector<uint64_t> kn, qn;
    host::gm_kq_levels(*p, Dist{mant, log2}, 1, kn, qn);
    *k_n = kn[0];
    *q_n = qn[0];
    return PRAND_OK;
}

extern "C" int prand_host_plan_sections(int gen, uint64_t length, uint64_t *n_sections, uint64_t *sec_len)
{
    if (gen < 0 || gen >= PRAND_NGEN) return PRAND_ERR_GEN;
    if (!n_sections || !sec_len || length == 0) return PRAND_ERR_ARG;
    plan_sections(gen, length, n_sections, sec_len);
    return PRAND_OK;
}

extern "C" int prand_host_plan_sections_sm(int gen, uint64_t length, int sm_count, uint64_t *n_sections, uint64_t *sec_len)
{
    if (gen < 0 || gen >= PRAND_NGEN) return PRAND_ERR_GEN;
    if (!n_sections || !sec_len || length == 0 || sm_count <= 0) return PRAND_ERR_ARG;
    plan_sections(gen, length, n_sections, sec_len, sm_count);
    return PRAND_OK;
}

extern "C" int prand_host_plan(int gen, uint64_t n_streams, uint64_t n_per_stream, int dtype, int sms,
                               uint64_t *chunk_len, uint64_t *n_chunks)
{
    if (gen < 0 || gen >= PRAND_NGEN) return PRAND_ERR_GEN;
    if (!chunk_len || !n_chunks || n_streams == 0 || dtype < 0 || dtype > 2 || sms <= 0) return PRAND_ERR_ARG;
    plan_chunks(gen, n_streams, n_per_stream, dtype, sms, chunk_len, n_chunks);
    return PRAND_OK;
}
