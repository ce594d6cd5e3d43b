// ris_boys_table.h -- host-side construction of the Boys interpolation tables used by ris_boys<M>
// (ris_core.cuh).  Row i (T0 = i/32): { e^{-T0}, c_0..c_6 },  c_k = (-1)^k F_{M+k}(T0) / k!.
// F_{M+6}(T0) from the convergent series  e^{-T} sum_k (2T)^k / [(2m+1)(2m+3)...(2m+2k+1)]
// in long double (all terms positive), lower orders by the downward recursion.
#pragma once
#include <cmath>
#include <vector>

inline void ris_build_boys_table(int M, int ngrid, int per_unit, std::vector<double>& out)
{
    const int top = M + 6;
    out.assign((size_t)ngrid * 8, 0.0);
    std::vector<long double> F(top + 1);
    for (int i = 0; i < ngrid; ++i) {
        const long double T = (long double)i / per_unit;
        const long double et = expl(-T);
        long double term = 1.0L / (2 * top + 1), sum = term;
        for (int k = 1; k < 4000; ++k) {
            term *= 2.0L * T / (2 * top + 2 * k + 1);
            sum += term;
            if (term < 1e-24L * sum) break;
        }
        F[top] = et * sum;
        for (int m = top - 1; m >= 0; --m) F[m] = (2.0L * T * F[m + 1] + et) / (2 * m + 1);
        double* row = &out[(size_t)i * 8];
        row[0] = (double)et;
        long double fact = 1.0L, sign = 1.0L;
        for (int k = 0; k <= 6; ++k) {
            if (k > 0) { fact *= k; sign = -sign; }
            row[1 + k] = (double)(sign * F[M + k] / fact);
        }
    }
}
