// tables.h -- host-side builders of the constant tables the kernels read (fp64 -> fp32 once).
#pragma once
#include <cmath>
#include <vector>
#include "fft_core.cuh"

namespace frs {

// per-thread stage twiddles: tw[(off_s + b*(R-1) + r-1)*P + p] = exp(-2 pi i ((p + b P) mod NS) r / (NS R))
inline std::vector<float2> build_twiddles(int n) {
    const int P = n / kE;
    std::vector<float2> tw((size_t)plan_tw_total(n) * P + 1);
    const double two_pi = 6.283185307179586476925286766559;
    for (int s = 1; s < plan_stages(n); ++s) {
        const int R = plan_radix(n, s), NB = kE / R, NS = plan_ns(n, s), off = plan_tw_off(n, s);
        for (int b = 0; b < NB; ++b)
            for (int r = 1; r < R; ++r)
                for (int p = 0; p < P; ++p) {
                    const int j = p + b * P;
                    const double ang = -two_pi * (double)((long long)(j % NS) * r) / (double)((long long)NS * R);
                    tw[(size_t)(off + b * (R - 1) + (r - 1)) * P + p] = make_float2((float)std::cos(ang), (float)std::sin(ang));
                }
    }
    return tw;
}

// twist[k] = exp(-2 pi i k / (2 n)), k = 0..n  (real<->complex packing, and the odd-bin shift of the
// zero-padded column transform)
inline std::vector<float2> build_twist(int n) {
    std::vector<float2> t(n + 1);
    const double pi = 3.1415926535897932384626433832795;
    for (int k = 0; k <= n; ++k) {
        const double ang = -pi * (double)k / (double)n;
        t[k] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    }
    return t;
}

}  // namespace frs
