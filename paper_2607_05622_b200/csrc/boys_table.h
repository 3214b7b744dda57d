// boys_table.h -- host-side generation of the Boys interpolation table used by the device evaluator (step a6).
// F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt is integrated directly with a composite 16-point Gauss-Legendre rule in
// long double (256 panels on [0,1]); the integrand is entire and, for T <= 36, varies on a scale >= 1/6, so the
// rule is exact to long-double round-off.  This is deliberately a different method from the CPU oracle's series.
#pragma once
#include <cmath>
#include <vector>

namespace ltjk {

inline void gauss_legendre(int n, std::vector<long double>& x, std::vector<long double>& w)
{
    x.assign(n, 0.0L); w.assign(n, 0.0L);
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < n; ++i) {
        long double z = std::cos(pi * (i + 0.75L) / (n + 0.5L)), pp = 0.0L;
        for (int it = 0; it < 100; ++it) {
            long double p1 = 1.0L, p2 = 0.0L;
            for (int j = 0; j < n; ++j) { long double p3 = p2; p2 = p1; p1 = ((2.0L * j + 1.0L) * z * p2 - j * p3) / (j + 1.0L); }
            pp = n * (z * p1 - p2) / (z * z - 1.0L);
            long double dz = p1 / pp;
            z -= dz;
            if (std::fabs((double)dz) < 1e-19) break;
        }
        x[i] = z; w[i] = 2.0L / ((1.0L - z * z) * pp * pp);
    }
}

// tab[i*nm + m] = F_m(i/8), i = 0..nt-1, m = 0..nm-1
inline std::vector<double> make_boys_table(int nt, int nm)
{
    std::vector<long double> gx, gw;
    gauss_legendre(16, gx, gw);
    const int npanel = 256;
    std::vector<double> tab((size_t)nt * nm);
    for (int i = 0; i < nt; ++i) {
        const long double T = (long double)i / 8.0L;
        std::vector<long double> acc(nm, 0.0L);
        for (int pnl = 0; pnl < npanel; ++pnl) {
            const long double a = (long double)pnl / npanel, h = 1.0L / npanel;
            for (int k = 0; k < 16; ++k) {
                const long double t = a + 0.5L * h * (gx[k] + 1.0L);
                const long double t2 = t * t;
                long double f = std::exp(-T * t2) * 0.5L * h * gw[k];
                for (int m = 0; m < nm; ++m) { acc[m] += f; f *= t2; }
            }
        }
        for (int m = 0; m < nm; ++m) tab[(size_t)i * nm + m] = (double)acc[m];
    }
    return tab;
}

}  // namespace ltjk
