// ssp_path.cu -- host-side path description for the screen generator: the Hufnagel-Valley 5/7 profile and the
// slab quantities the paper derives from it (PAPER.md:393 S21, :375 S18, :380 S19).  Plain double-precision
// host arithmetic (composite Simpson quadrature); no device work.  The outputs cn2[] / dz[] feed ssp_make_screens.
#include <cmath>
#include <vector>

#include "ssp_internal.h"

namespace {

double hv57(const ssp_hv57 *p, double h)
{
    const double gs = p->ground_scale > 0 ? p->ground_scale : 1000.0;   // as printed in S21 (textbook: 100 m)
    const double v = p->V / 27.0;
    return 0.00594 * v * v * pow(1e-5 * h, 10.0) * exp(-h / 1000.0) + 2.7e-16 * exp(-h / 1500.0) + p->A * exp(-h / gs);
}

template <class F>
double simpson(F f, double a, double b, int n) // n even
{
    const double h = (b - a) / n;
    double s = f(a) + f(b);
    for (int i = 1; i < n; ++i) s += f(a + i * h) * ((i & 1) ? 4.0 : 2.0);
    return s * h / 3.0;
}

// ---- screen placement ----------------------------------------------------------------------
// Piecewise-linear Cn2(z) through (zp[i], cp[i]); constant beyond the ends.
struct Profile {
    const double *zp, *cp;
    int n;
    double at(double z) const
    {
        if (z <= zp[0]) return cp[0];
        if (z >= zp[n - 1]) return cp[n - 1];
        int lo = 0, hi = n - 1;
        while (hi - lo > 1) {
            const int mid = (lo + hi) / 2;
            (zp[mid] <= z ? lo : hi) = mid;
        }
        return cp[lo] + (cp[hi] - cp[lo]) * (z - zp[lo]) / (zp[hi] - zp[lo]);
    }
    // sum over the linear pieces of [a, b] of  int (c0 + s (z - lo)) w(z) dz,  w = ((b - z)/(b - a))^p, p = 0 or 5/3,
    // each piece in closed form: with u = (b - z)/(b - a),  z - lo = (b - lo) - (b - a) u,
    //   piece = (b - a) [ (c0 + s (b - lo)) (u_lo^(p+1) - u_hi^(p+1))/(p+1) - s (b - a) (u_lo^(p+2) - u_hi^(p+2))/(p+2) ]
    double weighted(double a, double b, double p) const
    {
        const double d = b - a;
        if (!(d > 0)) return 0.0;
        double total = 0.0, lo = a;
        int i = 0;
        while (i < n && zp[i] <= a) ++i;                               // first kink strictly inside (a, ...)
        for (;;) {
            const double hi = (i < n && zp[i] < b) ? zp[i] : b;
            const double c0 = at(lo), c1 = at(hi);
            const double s = hi > lo ? (c1 - c0) / (hi - lo) : 0.0;
            const double ul = (b - lo) / d, uh = (b - hi) / d;
            total += d * ((c0 + s * (b - lo)) * (pow(ul, p + 1) - pow(uh, p + 1)) / (p + 1)
                          - s * d * (pow(ul, p + 2) - pow(uh, p + 2)) / (p + 2));
            if (hi >= b) break;
            lo = hi;
            ++i;
        }
        return total;
    }
};

struct Placer {
    Profile prof;
    double k76, limit;
    double rytov(double a, double b) const                              // S19 over [a, b], z from a
    {
        return b > a ? 3.27 * k76 * pow(b - a, 5.0 / 6.0) * prof.weighted(a, b, 5.0 / 3.0) : 0.0;
    }
};

constexpr int kMaxHalvings = 40;

} // namespace

extern "C" {

double ssp_dz_max(ssp_grid grid, double lambda, double n0)
{
    if (grid.N < 2 || !(grid.dx > 0) || !(lambda > 0) || !(n0 > 0)) return 0.0;
    const double pi = 3.14159265358979323846;
    const double k0 = 2.0 * pi / lambda, kap = pi / grid.dx;
    if (n0 * k0 <= kap) return 0.0;                                     // the grid carries evanescent frequencies
    return 0.5 * grid.N * grid.dx * sqrt(n0 * n0 * k0 * k0 - kap * kap) / kap;
}

int ssp_place_screens(const double *z_prof, const double *cn2_prof, int n_prof, const double *edges, int n_edges,
                      double lambda, double rytov_limit, double dz_max, int max_out, double *dz, double *cn2,
                      double *rytov, int *n_out)
{
    if (!z_prof || !cn2_prof || n_prof < 2 || !edges || n_edges < 2 || !(lambda > 0) || !(rytov_limit > 0) ||
        max_out < 1 || !dz || !cn2 || !n_out)
        return SSP_EINVAL;
    for (int i = 1; i < n_prof; ++i)
        if (!(z_prof[i] > z_prof[i - 1])) return SSP_EINVAL;
    for (int i = 1; i < n_edges; ++i)
        if (!(edges[i] > edges[i - 1])) return SSP_EINVAL;
    for (int i = 0; i < n_prof; ++i)
        if (!(cn2_prof[i] >= 0)) return SSP_EINVAL;
    const Placer P{{z_prof, cn2_prof, n_prof}, pow(2.0 * 3.14159265358979323846 / lambda, 7.0 / 6.0), rytov_limit};
    const size_t cap = (size_t)max_out * 4 + 16;                        // stages 1-2 may hold more pieces than the result
    std::vector<double> e;
    // 1. halve an interval until every piece is within the limit
    e.push_back(edges[0]);
    for (int q = 0; q + 1 < n_edges; ++q) {
        const double a = edges[q], b = edges[q + 1];
        long long parts = 1;
        for (int h = 0;; ++h) {
            bool ok = true;
            for (long long i = 0; i < parts && ok; ++i)
                ok = P.rytov(a + (b - a) * i / parts, a + (b - a) * (i + 1) / parts) <= rytov_limit;
            if (ok) break;
            if (h >= kMaxHalvings || (size_t)parts * 2 + e.size() > cap) return SSP_EUNSUPPORTED;
            parts *= 2;
        }
        for (long long i = 0; i < parts; ++i) e.push_back(a + (b - a) * (i + 1) / parts);
    }
    // 2. merge neighbours whose union stays within the limit, left to right
    for (size_t i = 0; i + 2 < e.size();) {
        if (P.rytov(e[i], e[i + 2]) <= rytov_limit) e.erase(e.begin() + i + 1);
        else ++i;
    }
    // 3. linear fit towards the limit, marching from the start
    std::vector<double> f{e[0]};
    {
        double a = e[0];
        size_t j = 1;
        const double end = e.back();
        for (;;) {
            double b1 = a, v1 = 0.0;
            while (j < e.size() && (e[j] <= a || P.rytov(a, e[j]) <= rytov_limit)) {
                if (e[j] > a) { b1 = e[j]; v1 = P.rytov(a, e[j]); }
                ++j;
            }
            if (j >= e.size()) {
                if (end > a) f.push_back(end);
                break;
            }
            const double b2 = e[j], v2 = P.rytov(a, b2);
            double step = (rytov_limit - v1) / (v2 - v1) * (b2 - b1);
            for (int h = 0; P.rytov(a, b1 + step) > rytov_limit; ++h) {
                if (h >= 200) return SSP_EUNSUPPORTED;
                step *= 0.5;
            }
            if (!(b1 + step > a) || f.size() > cap) return SSP_EUNSUPPORTED;
            a = b1 + step;
            f.push_back(a);
        }
    }
    // 4. halve an interval until it is no longer than the aliasing limit
    std::vector<double> g{f[0]};
    for (size_t q = 0; q + 1 < f.size(); ++q) {
        const double a = f[q], b = f[q + 1];
        long long parts = 1;
        for (int h = 0; dz_max > 0 && (b - a) / parts > dz_max; ++h) {
            if (h >= kMaxHalvings) return SSP_EUNSUPPORTED;
            parts *= 2;
        }
        if (g.size() + (size_t)parts > (size_t)max_out + 1) { *n_out = (int)(g.size() - 1 + parts); return SSP_EWORKSPACE; }
        for (long long i = 0; i < parts; ++i) g.push_back(a + (b - a) * (i + 1) / parts);
    }
    const int n = (int)g.size() - 1;
    for (int j = 0; j < n; ++j) {
        dz[j] = g[j + 1] - g[j];
        cn2[j] = P.prof.weighted(g[j], g[j + 1], 0.0) / dz[j];
        if (rytov) rytov[j] = P.rytov(g[j], g[j + 1]);
    }
    *n_out = n;
    return SSP_OK;
}

double ssp_hv57_cn2(const ssp_hv57 *p, double h) { return (p && h >= 0) ? hv57(p, h) : 0.0; }

int ssp_hv57_path(const ssp_hv57 *p, double h0, double L, int n, double lambda, double *cn2, double *dz,
                  double *rytov, double *r0)
{
    if (!p || !(h0 >= 0) || !(L > 0) || n < 1 || !(lambda > 0) || !cn2 || !dz) return SSP_EINVAL;
    const double k = 2.0 * 3.14159265358979323846 / lambda;
    const double d = L / n;
    double total = 0.0;
    for (int j = 0; j < n; ++j) {
        const double a = h0 + j * d;
        const double integral = simpson([&](double h) { return hv57(p, h); }, a, a + d, 1024);
        cn2[j] = integral / d;                                          // so that cn2[j] dz[j] is the S18 integral of the slab
        dz[j] = d;
        total += integral;
    }
    if (r0) *r0 = pow(0.423 * k * k * total, -3.0 / 5.0);              // S18 over the whole path
    if (rytov) {                                                        // S19, z measured from the source at h0
        const double w = simpson([&](double z) { return hv57(p, h0 + z) * pow(1.0 - z / L, 5.0 / 3.0); }, 0.0, L, 4096);
        *rytov = 3.27 * pow(k, 7.0 / 6.0) * pow(L, 5.0 / 6.0) * w;
    }
    return SSP_OK;
}

} // extern "C"
