// skip_ops.cpp -- host-side preparation of the skip operators; see skip_ops.h.
// Product code: shares nothing with oracle/.
#include "skip_ops.h"
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <dlfcn.h>
#include <mutex>
#include <string>

namespace prand {
namespace host {

typedef unsigned __int128 u128;

// ==================================================================================================
// LFSR113.  Component (p,q,s): with z = bits x_{ns}..x_{ns+31} (MSB first) the
// next word is made of bits s..p-1 of z followed by the recurrence bits x_{p+j} = x_j + x_{j+q}.
// ==================================================================================================
static const int LF_P[4] = {31, 29, 28, 25};
static const int LF_Q[4] = {6, 2, 13, 3};
static const int LF_S[4] = {18, 2, 7, 13};

uint32_t lfsr113_component_step(int c, uint32_t z)
{
    const int p = LF_P[c], q = LF_Q[c], s = LF_S[c];
    const uint32_t top_p = ~0u << (32 - p);
    uint32_t fresh = (z ^ (z << q)) >> (p - s);
    return ((z & top_p) << s) ^ fresh;
}

namespace {
struct Gf2Mat { uint32_t col[32]; };   // col[j] = image of 1u << j

inline uint32_t gf2_apply(const Gf2Mat &m, uint32_t v)
{
    uint32_t r = 0;
    while (v) {
        int j = __builtin_ctz(v);
        v &= v - 1;
        r ^= m.col[j];
    }
    return r;
}
inline Gf2Mat gf2_mul(const Gf2Mat &a, const Gf2Mat &b)   // a after b
{
    Gf2Mat r;
    for (int j = 0; j < 32; j++) r.col[j] = gf2_apply(a, b.col[j]);
    return r;
}
inline Gf2Mat gf2_identity()
{
    Gf2Mat r;
    for (int j = 0; j < 32; j++) r.col[j] = 1u << j;
    return r;
}

// generic: op^(mant) by right-to-left binary, then log2 squarings; Mul(a, b) must be associative
template <class Op, class Mul>
Op pow_dist(const Op &one_step, const Op &identity, Dist n, Mul mul)
{
    Op acc = identity, sq = one_step;
    for (uint64_t e = n.mant; e; e >>= 1) {
        if (e & 1) acc = mul(acc, sq);
        if (e >> 1) sq = mul(sq, sq);
    }
    for (unsigned i = 0; i < n.log2; i++) acc = mul(acc, acc);
    return acc;
}
}  // namespace

void lfsr113_levels(Dist n, unsigned levels, std::vector<LfsrOp> &out)
{
    out.assign(levels, LfsrOp());
    for (int c = 0; c < 4; c++) {
        Gf2Mat one;
        for (int j = 0; j < 32; j++) one.col[j] = lfsr113_component_step(c, 1u << j);
        Gf2Mat cur = pow_dist(one, gf2_identity(), n, gf2_mul);
        for (unsigned lev = 0; lev < levels; lev++) {
            std::memcpy(out[lev].col[c], cur.col, sizeof cur.col);
            if (lev + 1 < levels) cur = gf2_mul(cur, cur);
        }
    }
}

// ==================================================================================================
// MRG32K3A (eqs. 5-6)
// ==================================================================================================
namespace {
struct Mat3 { uint64_t e[9]; uint64_t mod; };

inline Mat3 mat3_mul(const Mat3 &a, const Mat3 &b)
{
    Mat3 r;
    r.mod = a.mod;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            uint64_t acc = 0;
            for (int l = 0; l < 3; l++) acc = (acc + a.e[3 * i + l] * b.e[3 * l + j] % a.mod) % a.mod;   // products < 2^64
            r.e[3 * i + j] = acc;
        }
    return r;
}
inline Mat3 mat3_identity(uint64_t mod)
{
    Mat3 r = {{1, 0, 0, 0, 1, 0, 0, 0, 1}, mod};
    return r;
}
}  // namespace

void mrg32k3a_levels(Dist n, unsigned levels, std::vector<MrgOp> &out)
{
    const uint64_t m1 = 4294967087ull, m2 = 4294944443ull;
    // X_{n+1} = A X_n on the column (x_n, x_{n-1}, x_{n-2}); negative coefficients as residues
    Mat3 A = {{0, 1403580ull, m1 - 810728ull, 1, 0, 0, 0, 1, 0}, m1};
    Mat3 B = {{527612ull, 0, m2 - 1370589ull, 1, 0, 0, 0, 1, 0}, m2};
    Mat3 a = pow_dist(A, mat3_identity(m1), n, mat3_mul);
    Mat3 b = pow_dist(B, mat3_identity(m2), n, mat3_mul);
    out.assign(levels, MrgOp());
    for (unsigned lev = 0; lev < levels; lev++) {
        for (int i = 0; i < 9; i++) {
            out[lev].a[i] = (uint32_t)a.e[i];
            out[lev].b[i] = (uint32_t)b.e[i];
        }
        if (lev + 1 < levels) { a = mat3_mul(a, a); b = mat3_mul(b, b); }
    }
}

// ==================================================================================================
// GM / GQ: the column (x(n), x(n-1)) advances by C = [[k, -q], [1, 0]] mod g.
// ==================================================================================================
namespace {
struct Mat2 { uint64_t e[4]; uint64_t g; };

inline uint64_t mulmod_g(uint64_t a, uint64_t b, uint64_t g) { return (uint64_t)((u128)a * b % g); }
inline Mat2 mat2_mul(const Mat2 &a, const Mat2 &b)
{
    Mat2 r;
    r.g = a.g;
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) {
            u128 t = (u128)mulmod_g(a.e[2 * i], b.e[j], a.g) + mulmod_g(a.e[2 * i + 1], b.e[2 + j], a.g);
            r.e[2 * i + j] = (uint64_t)(t % a.g);
        }
    return r;
}
inline Mat2 mat2_identity(uint64_t g)
{
    Mat2 r = {{1, 0, 0, 1}, g};
    return r;
}
inline Mat2 gm_companion(const GmParams &p)
{
    Mat2 c = {{p.k % p.g, (p.g - p.q % p.g) % p.g, 1, 0}, p.g};
    return c;
}
}  // namespace

void gm_levels(const GmParams &p, Dist n, unsigned levels, std::vector<GmOp> &out)
{
    Mat2 cur = pow_dist(gm_companion(p), mat2_identity(p.g), n, mat2_mul);
    out.assign(levels, GmOp());
    for (unsigned lev = 0; lev < levels; lev++) {
        for (int i = 0; i < 4; i++) out[lev].m[i] = cur.e[i];
        if (lev + 1 < levels) cur = mat2_mul(cur, cur);
    }
}

// The paper's own jump relation: x(2n+w) = k_n x(n+w) - q_n x(w) (eq. 2) with
// k_1 = k, q_1 = q, k_2n = k_n^2 - 2 q_n, q_2n = q_n^2 (eq. 3) and k_0 = 2, k_{n+1} = k k_n - q k_{n-1},
// q_n = q^n (eq. 4).  k_n is the Lucas sequence V_n(k, q); for an arbitrary n = mant * 2^log2 it is
// reached by the binary ladder on the pair (V_m, V_{m+1}) -- V_2m = V_m^2 - 2 q^m, V_2m+1 = V_m V_{m+1}
// - k q^m (both follow from eq. 2-4) -- over the bits of mant, then log2 doublings by eq. 3; further
// doublings give the levels n 2^j.  No matrix is involved: the CPU tests compare the result with the
// trace and determinant of the matrix power.
void gm_kq_levels(const GmParams &p, Dist n, unsigned levels, std::vector<uint64_t> &kn, std::vector<uint64_t> &qn)
{
    const uint64_t g = p.g, k = p.k % g, q = p.q % g;
    auto sub = [g](uint64_t a, uint64_t b) { return a >= b ? a - b : a + g - b; };
    // ladder over mant: (v0, v1, qm) = (V_m, V_{m+1}, q^m), m = leading bits of mant
    uint64_t v0 = 2 % g, v1 = k, qm = 1 % g;
    for (int b = 63; b >= 0; b--) {
        if (n.mant >> b == 0) continue;                   // above the leading bit: m stays 0
        const uint64_t v00 = sub(mulmod_g(v0, v0, g), mulmod_g(2 % g, qm, g));          // V_2m
        const uint64_t v01 = sub(mulmod_g(v0, v1, g), mulmod_g(k, qm, g));              // V_2m+1
        const uint64_t q2 = mulmod_g(qm, qm, g);
        if ((n.mant >> b) & 1) {
            const uint64_t v11 = sub(mulmod_g(v1, v1, g), mulmod_g(2 % g, mulmod_g(qm, q, g), g));   // V_2m+2
            v0 = v01; v1 = v11; qm = mulmod_g(q2, q, g);
        } else {
            v0 = v00; v1 = v01; qm = q2;
        }
    }
    uint64_t kc = v0, qc = qm;
    for (unsigned i = 0; i < n.log2; i++) {               // eq. 3
        kc = sub(mulmod_g(kc, kc, g), mulmod_g(2 % g, qc, g));
        qc = mulmod_g(qc, qc, g);
    }
    kn.assign(levels, 0);
    qn.assign(levels, 0);
    for (unsigned lev = 0; lev < levels; lev++) {
        kn[lev] = kc; qn[lev] = qc;
        kc = sub(mulmod_g(kc, kc, g), mulmod_g(2 % g, qc, g));
        qc = mulmod_g(qc, qc, g);
    }
}

bool gm_seed_state(const GmParams &p, uint64_t seed, uint64_t *words)
{
    const uint64_t w1 = seed % p.g;
    if (w1 == 0) return false;
    // D = C^(2^d); point i sits at orbit offset (i+1) 2^d: (w(n+1), w(n)) = C^n (w(1), w(0)) = C^n (w1, 0)
    Dist spacing = {1, p.d};
    Mat2 D = pow_dist(gm_companion(p), mat2_identity(p.g), spacing, mat2_mul);
    Mat2 cur = D;
    for (unsigned i = 0; i < p.s; i++) {
        words[2 * i] = mulmod_g(cur.e[2], w1, p.g);       // xP_i = w(n)
        words[2 * i + 1] = mulmod_g(cur.e[0], w1, p.g);   // xN_i = w(n+1)
        cur = mat2_mul(cur, D);
    }
    return true;
}

// ==================================================================================================
// MT19937.  Parameters of the paper's ref. [2] (reading T1):
// (w, n, m, r) = (32, 624, 397, 31), a = 0x9908B0DF.  Its characteristic polynomial has the closed
// form (ref. [2], appendix; w - r = 1 here)
//     phi(t) = u (v^31 + a_0 v^30 + ... + a_29 v + a_30) + a_31,   u = t^n + t^m, v = t^(n-1) + t^(m-1),
// a_i = bit i of a (a_31 is the most significant bit).  It is evaluated by Horner's rule in v with
// shift-and-xor products; prand_init self-checks it once per process (mt19937_phi_selfcheck below).
// ==================================================================================================
namespace {
constexpr int WIDE = 2 * MT_PW;                      // words of an unreduced product

inline void xor_shifted(uint64_t *dst, const uint64_t *src, int nwords, int shift_bits)
{
    const int ws = shift_bits >> 6, bs = shift_bits & 63;
    for (int i = 0; i < nwords; i++) {
        if (!src[i]) continue;
        dst[i + ws] ^= src[i] << bs;
        if (bs) dst[i + ws + 1] ^= src[i] >> (64 - bs);
    }
}

struct PhiData {
    MtPoly phi;
    std::vector<int> low_terms;                      // exponents of phi below the leading one
};

PhiData build_phi()
{
    const uint32_t a = 0x9908B0DFu;
    std::vector<uint64_t> h(WIDE + 2, 0), t(WIDE + 2, 0);
    h[0] = 1;
    for (int i = 0; i <= 30; i++) {                  // h = h v + a_i
        std::fill(t.begin(), t.end(), 0);
        xor_shifted(t.data(), h.data(), MT_PW, MT_N - 1);
        xor_shifted(t.data(), h.data(), MT_PW, MT_M - 1);
        if ((a >> i) & 1u) t[0] ^= 1;
        h.swap(t);
    }
    std::fill(t.begin(), t.end(), 0);                // phi = h u + a_31
    xor_shifted(t.data(), h.data(), MT_PW, MT_N);
    xor_shifted(t.data(), h.data(), MT_PW, MT_M);
    if ((a >> 31) & 1u) t[0] ^= 1;
    PhiData d;
    std::memcpy(d.phi.w, t.data(), sizeof d.phi.w);
    for (int e = 0; e < MT_DEG; e++)
        if ((d.phi.w[e >> 6] >> (e & 63)) & 1u) d.low_terms.push_back(e);
    return d;
}

const PhiData &phi_data()
{
    static const PhiData d = build_phi();
    return d;
}

// prod (WIDE words, degree <= 2*19936) -> prod mod phi in the low MT_PW words.  phi's second
// highest term is t^19710, so a 64-bit chunk of high coefficients folds strictly below itself.
void reduce_phi(uint64_t *prod)
{
    const std::vector<int> &terms = phi_data().low_terms;
    const int top_word = MT_DEG >> 6, top_bit = MT_DEG & 63;   // 311, 33
    for (int wi = WIDE - 1; wi >= top_word; wi--) {
        uint64_t H = prod[wi];
        if (wi == top_word) H &= ~0ull << top_bit;
        if (!H) continue;
        prod[wi] ^= H;
        const int base = wi * 64 - MT_DEG;
        for (size_t k = 0; k < terms.size(); k++) {
            int pos = base + terms[k];
            if (pos >= 0) {
                int ws = pos >> 6, bs = pos & 63;
                prod[ws] ^= H << bs;
                if (bs) prod[ws + 1] ^= H >> (64 - bs);
            } else {                                  // only for wi == top_word: chunk base below degree 0
                prod[0] ^= H >> (-pos);
            }
        }
    }
}

inline uint64_t spread32(uint32_t x)                  // bit i -> bit 2i
{
    uint64_t v = x;
    v = (v | (v << 16)) & 0x0000FFFF0000FFFFull;
    v = (v | (v << 8)) & 0x00FF00FF00FF00FFull;
    v = (v | (v << 4)) & 0x0F0F0F0F0F0F0F0Full;
    v = (v | (v << 2)) & 0x3333333333333333ull;
    v = (v | (v << 1)) & 0x5555555555555555ull;
    return v;
}
}  // namespace

const MtPoly &mt19937_phi() { return phi_data().phi; }

// phi(A) W = 0 (Cayley-Hamilton): sum over the set coefficients i of x_{i+j} must vanish for every word j >= 1 of
// a window and for the top bit of word 0.  Checked once per process on the sequence of seed 1; prand_init
// refuses MT19937 (PRAND_ERR_INTERNAL) if the closed form ever disagreed with the recurrence.
bool mt19937_phi_selfcheck()
{
    static const bool ok = [] {
        const PhiData &d = phi_data();
        std::vector<uint32_t> x(MT_DEG + MT_N + 1);
        mt19937_seed_state(1u, x.data());
        for (int k = 0; k + MT_N < (int)x.size(); k++) {
            const uint32_t y = (x[k] & 0x80000000u) | (x[k + 1] & 0x7FFFFFFFu);
            x[k + MT_N] = x[k + MT_M] ^ (y >> 1) ^ ((y & 1u) ? 0x9908B0DFu : 0u);
        }
        for (int j = 0; j < 4; j++) {
            uint32_t acc = x[MT_DEG + j];                  // leading coefficient
            for (int e : d.low_terms) acc ^= x[e + j];
            if (j == 0) acc &= 0x80000000u;                // only the top bit of word 0 is state
            if (acc) return false;
        }
        return true;
    }();
    return ok;
}

void mt19937_sqrmod(MtPoly &r, const MtPoly &a)
{
    uint64_t prod[WIDE + 2];
    for (int i = 0; i < MT_PW; i++) {
        prod[2 * i] = spread32((uint32_t)a.w[i]);
        prod[2 * i + 1] = spread32((uint32_t)(a.w[i] >> 32));
    }
    prod[WIDE] = prod[WIDE + 1] = 0;
    reduce_phi(prod);
    std::memcpy(r.w, prod, sizeof r.w);
}

// 4-bit comb: T[c] = c(x) b(x) for the 16 polynomials c of degree < 4; the nibbles of a are
// consumed from the most significant nibble position down, shifting the accumulator by 4 between.
void mt19937_mulmod(MtPoly &r, const MtPoly &a, const MtPoly &b)
{
    static thread_local uint64_t T[16][MT_PW + 1];
    std::memset(T, 0, sizeof T);
    for (int c = 1; c < 16; c++) {
        if (c & (c - 1)) {                            // composite: lowest set bit + rest
            int low = c & -c;
            for (int i = 0; i <= MT_PW; i++) T[c][i] = T[low][i] ^ T[c ^ low][i];
        } else {
            int sh = __builtin_ctz(c);
            for (int i = 0; i < MT_PW; i++) {
                T[c][i] ^= b.w[i] << sh;
                if (sh) T[c][i + 1] ^= b.w[i] >> (64 - sh);
            }
        }
    }
    uint64_t prod[WIDE + 2];
    std::memset(prod, 0, sizeof prod);
    for (int nib = 15; nib >= 0; nib--) {
        for (int j = 0; j < MT_PW; j++) {
            unsigned c = (unsigned)(a.w[j] >> (4 * nib)) & 15u;
            if (!c) continue;
            for (int i = 0; i <= MT_PW; i++) prod[j + i] ^= T[c][i];
        }
        if (nib) {
            for (int i = WIDE + 1; i > 0; i--) prod[i] = (prod[i] << 4) | (prod[i - 1] >> 60);
            prod[0] <<= 4;
        }
    }
    reduce_phi(prod);
    std::memcpy(r.w, prod, sizeof r.w);
}

// ---- the precomputed table ------------------------------------------------------------
namespace {
std::vector<MtPoly> g_table;
bool g_table_tried = false;
std::mutex g_table_mu;

std::string table_path()
{
    if (const char *env = std::getenv("PRAND_MT_TABLE")) return env;
    Dl_info info;
    if (dladdr((const void *)&mt19937_seed_state, &info) && info.dli_fname) {
        std::string p = info.dli_fname;
        const size_t slash = p.rfind('/');
        return (slash == std::string::npos ? std::string(".") : p.substr(0, slash)) + "/mt19937_polys.bin";
    }
    return "mt19937_polys.bin";
}
// A table of the right size can still be stale (another record layout) or damaged, and would silently give wrong
// block-split streams.  Every record is the square of its predecessor in its chain (x^(2^n); x^(m 2^i) for each m), the
// chains meet at x^16 = record (m = 16, i = 0) = record (2^4), and x^m is a product of the first records: checking the
// head, some middle links and the tail of every chain with the host's own polynomial arithmetic costs ~50 squarings
// once per process and catches a wrong layout, a truncated-and-padded file and most bit damage.
bool table_consistent(const std::vector<MtPoly> &t)
{
    auto same = [](const MtPoly &a, const MtPoly &b) { return std::memcmp(a.w, b.w, sizeof a.w) == 0; };
    MtPoly r;
    for (int n : {1, 2, 3, 4, 17, 100, 255, 256, MT_TABLE_POW2 - 1}) {
        mt19937_sqrmod(r, t[n - 1]);
        if (!same(r, t[n])) return false;
    }
    for (int m = MT_TABLE_M0; m <= MT_TABLE_M1; m++) {
        const MtPoly *row = t.data() + MT_TABLE_POW2 + (m - MT_TABLE_M0) * MT_TABLE_SHIFTS;
        MtPoly xm;                                            // x^m from the bits of m
        bool first = true;
        for (int b = 0; b < 5; b++) {
            if (!((m >> b) & 1)) continue;
            if (first) { xm = t[b]; first = false; }
            else mt19937_mulmod(xm, xm, t[b]);
        }
        if (!same(xm, row[0])) return false;
        for (int i : {1, 64, MT_TABLE_SHIFTS - 1}) {
            mt19937_sqrmod(r, row[i - 1]);
            if (!same(r, row[i])) return false;
        }
    }
    return true;
}
}  // namespace

const MtPoly *mt19937_table()
{
    if (prand::debug_hooks().mt_host_poly) return nullptr;     // hook: every polynomial by host arithmetic
    std::lock_guard<std::mutex> lock(g_table_mu);
    if (!g_table_tried) {
        g_table_tried = true;
        if (FILE *f = std::fopen(table_path().c_str(), "rb")) {
            std::vector<MtPoly> t(MT_TABLE_ENTRIES);
            const size_t n = std::fread(t.data(), sizeof(MtPoly), t.size(), f);
            char extra;
            const bool exact = n == t.size() && std::fread(&extra, 1, 1, f) == 0;
            std::fclose(f);
            // record 0 must be the polynomial x, record 1 x^2: a cheap guard against a foreign file
            if (exact && t[0].w[0] == 2 && t[1].w[0] == 4) {
                if (table_consistent(t)) g_table.swap(t);
                else std::fprintf(stderr, "libprand: %s fails its consistency check (stale or damaged file); MT19937 jump "
                                          "polynomials are computed on the host instead\n", table_path().c_str());
            }
        }
    }
    return g_table.empty() ? nullptr : g_table.data();
}

int mt19937_table_index(Dist v)
{
    if (v.mant == 0) return -1;
    const unsigned tz = (unsigned)__builtin_ctzll(v.mant);
    const uint64_t odd = v.mant >> tz;
    const uint64_t log2 = (uint64_t)v.log2 + tz;
    if (odd == 1) return log2 < (uint64_t)MT_TABLE_POW2 ? (int)log2 : -1;
    // m 2^i with m in 15..24: m = odd 2^k for some k <= 4 taken from the power of two
    for (unsigned k = 0; k <= 4 && k <= log2; k++) {
        const uint64_t m = odd << k;
        if (m > (uint64_t)MT_TABLE_M1) break;
        if (m >= (uint64_t)MT_TABLE_M0 && log2 - k < (uint64_t)MT_TABLE_SHIFTS)
            return MT_TABLE_POW2 + (int)(m - MT_TABLE_M0) * MT_TABLE_SHIFTS + (int)(log2 - k);
    }
    return -1;
}

bool mt19937_table_terms(Dist v, std::vector<int> &idx)
{
    idx.clear();
    const int whole = mt19937_table_index(v);
    if (whole >= 0) { idx.push_back(whole); return true; }
    for (uint64_t e = v.mant; e; e &= e - 1) {
        const uint64_t n = (uint64_t)__builtin_ctzll(e) + v.log2;
        if (n >= (uint64_t)MT_TABLE_POW2) { idx.clear(); return false; }
        idx.push_back((int)n);
    }
    return true;
}

void mt19937_xpow(Dist n, MtPoly &out)
{
    // tabulated distances cost a copy; sums of tabulated distances one product per extra term
    std::vector<int> idx;
    const MtPoly *t = mt19937_table();
    if (t && n.mant && mt19937_table_terms(n, idx) && idx.size() <= 8) {
        out = t[idx[0]];
        for (size_t k = 1; k < idx.size(); k++) mt19937_mulmod(out, out, t[idx[k]]);
        return;
    }
    mt19937_xpow_raw(n, out);
}

void mt19937_xpow_raw(Dist n, MtPoly &out)
{
    MtPoly acc;
    std::memset(&acc, 0, sizeof acc);
    if (n.mant == 0) { acc.w[0] = 1; out = acc; return; }   // x^0
    // left-to-right over mant: square, then multiply by x (a one-bit shift and one fold)
    acc.w[0] = 1;
    for (int b = 63 - __builtin_clzll(n.mant); b >= 0; b--) {
        mt19937_sqrmod(acc, acc);
        if ((n.mant >> b) & 1u) {
            uint64_t prod[WIDE + 2];
            std::memset(prod, 0, sizeof prod);
            xor_shifted(prod, acc.w, MT_PW, 1);
            reduce_phi(prod);
            std::memcpy(acc.w, prod, sizeof acc.w);
        }
    }
    for (unsigned i = 0; i < n.log2; i++) mt19937_sqrmod(acc, acc);
    out = acc;
}

// PRAND ships its jump polynomials precomputed because each costs milliseconds of serial host work
// (PAPER.md:378).  Here they are computed on demand and the ladder x^(n 2^j) mod phi of the most
// recent distances is kept, so that a second prand_init / prand_jump with the same distance (a
// bench step, a family of shards) costs a copy.
void mt19937_levels(Dist n, unsigned levels, std::vector<MtPoly> &out)
{
    struct Entry { Dist n; std::vector<MtPoly> ladder; };
    static std::mutex mu;
    static std::vector<Entry> cache;                       // most recently used last, at most 8 distances
    out.assign(levels, MtPoly());
    if (!levels) return;
    std::lock_guard<std::mutex> lock(mu);
    size_t hit = cache.size();
    for (size_t i = 0; i < cache.size(); i++)
        if (cache[i].n.mant == n.mant && cache[i].n.log2 == n.log2) hit = i;
    if (hit == cache.size()) {
        if (cache.size() == 8) cache.erase(cache.begin());
        cache.push_back(Entry{n, std::vector<MtPoly>(1)});
        mt19937_xpow(n, cache.back().ladder[0]);
        hit = cache.size() - 1;
    }
    std::vector<MtPoly> &lad = cache[hit].ladder;
    const MtPoly *table = mt19937_table();
    while (lad.size() < levels) {
        lad.emplace_back();
        const Dist d = {n.mant, n.log2 + (unsigned)(lad.size() - 1)};
        const int ti = table && n.mant ? mt19937_table_index(d) : -1;
        if (ti >= 0) lad.back() = table[ti];
        else mt19937_sqrmod(lad[lad.size() - 1], lad[lad.size() - 2]);
    }
    for (unsigned lev = 0; lev < levels; lev++) out[lev] = lad[lev];
}

void mt19937_to_op(const MtPoly &p, MtOp &op)
{
    for (int i = 0; i < MT_PW; i++) {
        op.w[2 * i] = (uint32_t)p.w[i];
        op.w[2 * i + 1] = (uint32_t)(p.w[i] >> 32);
    }
}

void mt19937_seed_state(uint32_t seed, uint32_t *w)
{
    w[0] = seed;
    for (uint32_t i = 1; i < (uint32_t)MT_N; i++) {
        uint32_t prev = w[i - 1];
        w[i] = 1812433253u * (prev ^ (prev >> 30)) + i;
    }
}

}  // namespace host
}  // namespace prand
