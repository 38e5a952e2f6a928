// tables.h -- host-side builders of the constant tables the kernels read (fp64 -> fp32 once).
#pragma once
#include <cmath>
#include <vector>
#include "fft_core.cuh"
#include "fft_dif.cuh"

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

// twiddles of the DIF/DIT core (fft_dif.cuh): direct table of tw2, factorised base of tw1
template <int N>
inline std::vector<float4> build_dif_twiddles() {
    using D = Dif<N>;
    std::vector<float4> tw((size_t)D::TW_TOTAL, make_float4(1.f, 0.f, 1.f, 0.f));
    const double two_pi = 6.283185307179586476925286766559;
    auto ex = [&](long long num, long long den) {
        const double ang = -two_pi * (double)num / (double)den;
        return make_float2((float)std::cos(ang), (float)std::sin(ang));
    };
    if (D::C > 1)
        for (int q = 0; q < 8; ++q)
            for (int n0 = 0; n0 < D::C; ++n0) {
                const float2 w1 = ex((long long)n0 * (2 * q + 1), 16LL * D::C);
                const float2 w2 = 2 * q + 2 < kE ? ex((long long)n0 * (2 * q + 2), 16LL * D::C) : make_float2(1.f, 0.f);
                tw[(size_t)q * D::C + n0] = make_float4(w1.x, w1.y, w2.x, w2.y);
            }
    float2* f = reinterpret_cast<float2*>(tw.data() + D::TW_D);
    for (int a = 0; a < D::C; ++a) f[a] = ex(16LL * a, N);
    for (int c = 0; c < 16; ++c) f[D::C + c] = ex(c, N);
    return tw;
}
inline std::vector<float4> build_dif_twiddles(int n) {
    switch (n) {
        case 256: return build_dif_twiddles<256>();
        case 512: return build_dif_twiddles<512>();
        case 1024: return build_dif_twiddles<1024>();
        case 2048: return build_dif_twiddles<2048>();
        case 4096: return build_dif_twiddles<4096>();
        default: return {};
    }
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
