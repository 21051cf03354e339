// mt_table_gen.cpp -- build step: writes the MT19937 jump-polynomial table of PAPER.md:378 (section 5.4).
//
// "In PRAND the coefficients are already calculated for the following values of v: v = 2^n, n = 0..511 and
// v = n 2^i, n = 15..24, i = 0..127.  Coefficients of each polynomial require 2496 bytes in memory,
// therefore, less than 5 megabytes are needed."  This program computes exactly those 512 + 1280 polynomials
// g_v(x) = x^v mod phi(x) with the library's own host arithmetic (skip_ops.cpp: sparse phi, squaring by bit
// spreading) and writes them as 1792 records of 312 little-endian 64-bit words (bit (i & 63) of word i >> 6 =
// coefficient of x^i): record n for 2^n, record 512 + 128 (m - 15) + i for m 2^i.  paper_1307_5869_b200/build.py
// runs it once; libprand loads the file at run time (skip_ops.cpp), keeps it resident on the device and then
// needs no polynomial arithmetic for block lengths and jump distances of these forms.
// Usage: mt_table_gen OUT.bin
#include <cstdio>
#include <vector>
#include "skip_ops.h"

using namespace prand::host;

// the generator computes everything by square-and-multiply: no table exists yet
namespace prand {
const DebugHooks &debug_hooks()
{
    static DebugHooks h = {};
    h.mt_host_poly = true;
    return h;
}
}  // namespace prand

int main(int argc, char **argv)
{
    if (argc != 2) { std::fprintf(stderr, "usage: %s OUT.bin\n", argv[0]); return 2; }
    std::vector<MtPoly> table(MT_TABLE_ENTRIES);
    mt19937_xpow_raw(Dist{1, 0}, table[0]);
    for (int n = 1; n < MT_TABLE_POW2; n++) mt19937_sqrmod(table[n], table[n - 1]);
    for (int m = MT_TABLE_M0; m <= MT_TABLE_M1; m++) {
        MtPoly *row = &table[MT_TABLE_POW2 + (m - MT_TABLE_M0) * MT_TABLE_SHIFTS];
        mt19937_xpow_raw(Dist{(uint64_t)m, 0}, row[0]);
        for (int i = 1; i < MT_TABLE_SHIFTS; i++) mt19937_sqrmod(row[i], row[i - 1]);
    }
    FILE *f = std::fopen(argv[1], "wb");
    if (!f) { std::perror(argv[1]); return 1; }
    const size_t n = std::fwrite(table.data(), sizeof(MtPoly), table.size(), f);
    if (std::fclose(f) != 0 || n != table.size()) { std::fprintf(stderr, "short write\n"); return 1; }
    return 0;
}
