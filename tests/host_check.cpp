// host_check.cpp -- TEST-ONLY host build of the generated OS/HGP recurrences and the Boys evaluator.
// Compiled with g++ into libltjk_hostcheck.so by tests (never linked into libltjk.so, never used by the product
// path): it lets the CPU test tier check the code generator against the oracle before any GPU time is spent.
#include "eri_core.h"
#include "boys_table.h"
#include <cstring>

using namespace ltjk;

static const double* table()
{
    static std::vector<double> t = make_boys_table(kBoysNT, kBoysNM);
    return t.data();
}

template <int LA, int LB, int LC, int LD>
static void run(const double* bra, const double* ket, double* out) { eri_quartet<LA, LB, LC, LD>(bra, ket, table(), out); }

typedef void (*fn_t)(const double*, const double*, double*);

template <int CB, int CK> struct Disp {
    static fn_t get() {
        constexpr int la[6] = {0, 1, 1, 2, 2, 2}, lb[6] = {0, 0, 1, 0, 1, 2};
        return &run<la[CB], lb[CB], la[CK], lb[CK]>;
    }
};

template <int CB, int CK> static void fill(fn_t (*t)[6]) {
    if constexpr (CK <= CB) t[CB][CK] = Disp<CB, CK>::get();
    if constexpr (CK < 5) fill<CB, CK + 1>(t);
    else if constexpr (CB < 5) fill<CB + 1, 0>(t);
}

static int pair_class(int la, int lb) { return la * (la + 1) / 2 + lb; }

extern "C" {

// shells given as (centre[3], l, nprim, exps, coefs); requires la>=lb, lc>=ld.  If braclass < ketclass the roles are
// swapped internally and the output is transposed back, exactly as the device kernel does.
int hc_eri_quartet(const double* A, int la, int na, const double* ea, const double* ca,
                   const double* B, int lb, int nb, const double* eb, const double* cb,
                   const double* C, int lc, int nc, const double* ec, const double* cc,
                   const double* D, int ld, int nd, const double* ed, const double* cd, double* out)
{
    static fn_t tab[6][6];
    static bool init = false;
    if (!init) { memset(tab, 0, sizeof(tab)); fill<0, 0>(tab); init = true; }
    if (la < lb || lc < ld || la > 2 || lc > 2) return -1;
    double bra[kPairStride], ket[kPairStride];
    build_pair_record(A, B, na, ea, ca, nb, eb, cb, bra);
    build_pair_record(C, D, nc, ec, cc, nd, ed, cd, ket);
    const int cbr = pair_class(la, lb), ckt = pair_class(lc, ld);
    const int nab = ncart(la) * ncart(lb), ncd = ncart(lc) * ncart(ld);
    if (cbr >= ckt) {
        tab[cbr][ckt](bra, ket, out);
    } else {
        std::vector<double> tmp((size_t)nab * ncd);
        tab[ckt][cbr](ket, bra, tmp.data());
        for (int i = 0; i < nab; ++i) for (int j = 0; j < ncd; ++j) out[i * ncd + j] = tmp[(size_t)j * nab + i];
    }
    return 0;
}

void hc_boys(int mmax, double T, double* F)
{
    switch (mmax) {
    case 0: boys_scaled<0>(T, 1.0, table(), F); break;
    case 1: boys_scaled<1>(T, 1.0, table(), F); break;
    case 2: boys_scaled<2>(T, 1.0, table(), F); break;
    case 3: boys_scaled<3>(T, 1.0, table(), F); break;
    case 4: boys_scaled<4>(T, 1.0, table(), F); break;
    case 5: boys_scaled<5>(T, 1.0, table(), F); break;
    case 6: boys_scaled<6>(T, 1.0, table(), F); break;
    case 7: boys_scaled<7>(T, 1.0, table(), F); break;
    default: boys_scaled<8>(T, 1.0, table(), F); break;
    }
}

}
