// ssp_path.cu -- host-side path description for the screen generator: the Hufnagel-Valley 5/7 profile and the
// slab quantities the paper derives from it (PAPER.md:393 S21, :375 S18, :380 S19).  Plain double-precision
// host arithmetic (composite Simpson quadrature); no device work.  The outputs cn2[] / dz[] feed ssp_make_screens.
#include <cmath>

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

} // namespace

extern "C" {

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
