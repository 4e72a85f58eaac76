// pm_growth.cu -- host-side fp64 scalars of the time integrator (no device code).
//
// PAPER.md App. A (L516-555) defines the linear growth D1 by the ODE A1 and the FastPM factors by
// G_D = a^2 dD1/dt, G_K = a dG_D/dt (eq. A7; eq. 14-15).  For flat matter + Lambda the
// growing solution of A1 normalised to D1 -> a in matter domination (A3, L528) has the closed-form
// quadrature (Heath 1977)
//     D1(a) = 5/2 Om E(a) I(a),   I(a) = int_0^a da' / (a' E(a'))^3,   E^2 = Om a^-3 + 1 - Om,
// which this file evaluates directly (the oracle integrates the ODE instead: two routes, one answer).
//     dD1/da = 5/2 Om [E'(a) I(a) + E / (a E)^3],  E' = -3/2 Om a^-4 / E
//     G_D = a^2 H dD1/dlna = a^3 E dD1/da                  (H0 = 1)
//     G_K = 3/2 Om D1                                      (A7 with A1 substituted for D1'')
#include <cmath>

#include "pm_internal.cuh"

namespace pm {

static double heath_integral(double om, double a)
{
    // substitute u = sqrt(a'): integrand 2 u^4 (Om + (1-Om) u^6)^-3/2 is smooth on [0, sqrt(a)]
    const int n = 8192;  // composite Simpson
    const double U = std::sqrt(a), h = U / n, ol = 1.0 - om;
    auto f = [&](double u) {
        double u2 = u * u, u6 = u2 * u2 * u2;
        double b = om + ol * u6;
        return 2.0 * u2 * u2 / (b * std::sqrt(b));
    };
    double sum = f(0.0) + f(U);
    for (int i = 1; i < n; i++) sum += f(h * i) * ((i & 1) ? 4.0 : 2.0);
    return sum * h / 3.0;
}

void growth_host(double om, double a, double out[4])
{
    double E2 = om / (a * a * a) + 1.0 - om, E = std::sqrt(E2);
    double I = heath_integral(om, a);
    double D1 = 2.5 * om * E * I;
    double dE = -1.5 * om / (a * a * a * a) / E;
    double aE = a * E;
    double dD1da = 2.5 * om * (dE * I + E / (aE * aE * aE));
    out[0] = D1;
    out[1] = a * dD1da;
    out[2] = a * a * a * E * dD1da;
    out[3] = 1.5 * om * D1;
}

// eq. 15 (L165): D(tc, ta, tb) = (D1(tb) - D1(ta)) / G_D(tc); antisymmetric in (ta, tb) bit for bit
double drift_factor_host(double om, double ac, double aa, double ab)
{
    double gb[4], ga[4], gc[4];
    growth_host(om, ab, gb);
    growth_host(om, aa, ga);
    growth_host(om, ac, gc);
    return (gb[0] - ga[0]) / gc[2];
}

// eq. 15 (L167): K(tc, ta, tb) = (G_D(tb) - G_D(ta)) / G_K(tc)
double kick_factor_host(double om, double ac, double aa, double ab)
{
    double gb[4], ga[4], gc[4];
    growth_host(om, ab, gb);
    growth_host(om, aa, ga);
    growth_host(om, ac, gc);
    return (gb[2] - ga[2]) / gc[3];
}

}  // namespace pm
