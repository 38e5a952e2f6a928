// tables.h -- host-side builders of the constant tables the kernels read (fp64 -> fp32 once).
#pragma once
#include <cmath>
#include <vector>
#include "fft_core.cuh"

namespace frs {

// packed stage twiddles, layout of fft_core.cuh plan_tw_* (direct or factorised per stage)
inline std::vector<float4> build_twiddles(int n) {
    std::vector<float4> tw((size_t)plan_tw_total(n), make_float4(1.f, 0.f, 1.f, 0.f));
    const double two_pi = 6.283185307179586476925286766559;
    auto ex = [&](long long num, long long den) {
        const double ang = -two_pi * (double)num / (double)den;
        return make_float2((float)std::cos(ang), (float)std::sin(ang));
    };
    for (int s = 1; s < plan_stages(n); ++s) {
        const int R = plan_radix(n, s), NS = plan_ns(n, s), off = plan_tw_off(n, s), HP = R / 2, WA = plan_tw_wa(n, s);
        const long long den = (long long)NS * R;
        if (plan_tw_fact(n, s)) {
            float2* f = reinterpret_cast<float2*>(tw.data() + off);
            for (int a = 0; a < WA; ++a) f[a] = ex(16LL * a, den);
            for (int c = 0; c < 16; ++c) f[WA + c] = ex(c, den);
        } else {
            for (int q = 0; q < HP; ++q)
                for (int j = 0; j < WA; ++j) {
                    const int r1 = 2 * q + 1, r2 = 2 * q + 2;
                    const float2 w1 = ex((long long)j * r1, den), w2 = r2 < R ? ex((long long)j * r2, den) : make_float2(1.f, 0.f);
                    tw[(size_t)off + q * WA + j] = make_float4(w1.x, w1.y, w2.x, w2.y);
                }
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
