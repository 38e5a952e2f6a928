// selftest.cu -- CPU replay of the register/shared-memory FFT logic of fft_core.cuh, thread by
// thread, with the "shared memory" exchange emulated by a host array.  Lets the index maps, plans
// and twiddle tables be tested where there is no GPU (tests/test_host_logic.py).
#include <vector>
#include "../../include/frs.h"
#include "fft_core.cuh"
#include "tables.h"
#include "tmap.h"

namespace frs {
struct Regs { C2 v[kE]; };

// pair (a, b = 2a) through the float4 exchange path the kernels use
template <int N, bool INV, int S>
static void emu_from(std::vector<Regs>& regs, std::vector<float4>& buf, const float4* tw) {
    constexpr int P = N / kE;
    if constexpr (S < plan_stages(N)) {
        for (int p = 0; p < P; ++p) stage_compute<N, S, INV>(regs[p].v, p, tw);
        if constexpr (S + 1 < plan_stages(N)) {
            for (int p = 0; p < P; ++p) stage_scatter2<N, S>(regs[p].v, p, buf.data());
            for (int p = 0; p < P; ++p) canon_gather2<N>(regs[p].v, p, buf.data());
        }
        emu_from<N, INV, S + 1>(regs, buf, tw);
    }
}
template <int N>
static int emu(int inverse, const float2* in, float2* out) {
    constexpr int P = N / kE;
    std::vector<float4> tw = build_twiddles(N);
    std::vector<Regs> regs(P);
    std::vector<float4> buf(xbuf_len(N));
    for (int p = 0; p < P; ++p)
        for (int e = 0; e < kE; ++e) {
            regs[p].v[e] = c2make(in[p + e * P], cscale(in[p + e * P], 2.0f));
        }
    if (inverse) emu_from<N, true, 0>(regs, buf, tw.data());
    else emu_from<N, false, 0>(regs, buf, tw.data());
    int bad = 0;
    for (int p = 0; p < P; ++p)
        for (int e = 0; e < kE; ++e) {
            const float2 a = c2get(regs[p].v[e], 0), b = c2get(regs[p].v[e], 1);
            out[p + e * P] = a;
            if (b.x != 2.0f * a.x || b.y != 2.0f * a.y) bad = 1;     // scaling by 2 is exact in fp32
        }
    return bad ? FRS_ESTATE : 0;
}
}  // namespace frs

// ---- DIF/DIT core (fft_dif.cuh) ----------------------------------------------------------------------
namespace frs {
// forward: natural time order in, natural frequency order out (the permuted spectrum is sorted here);
// inverse: natural frequency order in (placed in the permuted layout), natural time order out.
template <int N>
static int emu_dif(int inverse, const float2* in, float2* out) {
    using D = Dif<N>;
    constexpr int P = D::P;
    std::vector<float4> tw = build_dif_twiddles<N>();
    std::vector<Regs> regs(P);
    std::vector<float4> X(D::XLEN);
    int bad = 0;
    if (!inverse) {
        for (int t = 0; t < P; ++t)
            for (int e = 0; e < kE; ++e) regs[t].v[e] = c2make(in[t + e * P], cscale(in[t + e * P], 2.0f));
        for (int t = 0; t < P; ++t) dif_fwd_0<N>(regs[t].v, t, X.data(), tw.data());
        for (int t = 0; t < P; ++t) dif_fwd_1<N>(regs[t].v, t, X.data(), tw.data());
        for (int t = 0; t < P; ++t) dif_fwd_2<N>(regs[t].v, t, X.data());
        for (int t = 0; t < P; ++t)
            for (int e = 0; e < kE; ++e) {
                const float2 a = c2get(regs[t].v[e], 0), b = c2get(regs[t].v[e], 1);
                out[D::freq_index(t, e)] = a;
                if (b.x != 2.0f * a.x || b.y != 2.0f * a.y) bad = 1;
            }
    } else {
        for (int t = 0; t < P; ++t)
            for (int e = 0; e < kE; ++e) {
                const float2 a = in[D::freq_index(t, e)];
                regs[t].v[e] = c2make(a, cscale(a, 2.0f));
            }
        for (int t = 0; t < P; ++t) dif_inv_0<N>(regs[t].v, t, X.data());
        for (int t = 0; t < P; ++t) dif_inv_1<N>(regs[t].v, t, X.data(), tw.data());
        for (int t = 0; t < P; ++t) dif_inv_2<N>(regs[t].v, t, X.data(), tw.data());
        for (int t = 0; t < P; ++t)
            for (int e = 0; e < kE; ++e) {
                const float2 a = c2get(regs[t].v[e], 0), b = c2get(regs[t].v[e], 1);
                out[t + e * P] = a;
                if (b.x != 2.0f * a.x || b.y != 2.0f * a.y) bad = 1;
            }
    }
    return bad ? FRS_ESTATE : 0;
}

// Race and bank-conflict analysis of the exchange pattern, lane by lane (what racecheck would look at).
// Program order of one column after another:  put_time | BLOCK | get_mid put_mid | WARP | get_freq  put_freq | WARP |
// get_mid put_mid | BLOCK | get_time  put_time (next column) ...   (no synchronisation where there is only a space)
template <int N>
static int dif_exchange_report(int* out) {
    using D = Dif<N>;
    constexpr int P = D::P;
    enum Kind { kTime = 0, kMid = 1, kFreq = 2 };
    struct Acc { int epoch, thread; bool write; };
    struct Step { int kind; bool write; int sync_after; };       // sync_after: 0 none, 1 warp, 2 block
    const Step cycle[] = {{kTime, true, 2}, {kMid, false, 0}, {kMid, true, 1}, {kFreq, false, 0}, {kFreq, true, 1},
                          {kMid, false, 0}, {kMid, true, 2}, {kTime, false, 0}};
    auto slot = [&](int kind, int t, int i) {
        return kind == kTime ? D::base_time(t) + D::off_time(i) : kind == kMid ? D::base_mid(t) + D::off_mid(i)
                                                                              : D::base_freq(t) + D::off_freq(i);
    };
    const bool three = D::C > 1;
    std::vector<std::vector<Acc>> log(D::XLEN);
    std::vector<int> sync_kind;                                  // sync that ends epoch e
    int epoch = 0, oob = 0, worst_conflict = 1;
    for (int rep = 0; rep < 2; ++rep)
        for (const Step& st : cycle) {
            if (!three && (st.kind == kFreq || (st.kind == kMid && ((st.write && st.sync_after == 1) || (!st.write && &st == &cycle[5])))))
                continue;                                        // two-stage transform: no X2
            for (int t = 0; t < P; ++t)
                for (int i = 0; i < kE; ++i) {
                    const int s = slot(st.kind, t, i);
                    if (s < 0 || s >= D::XLEN) { ++oob; continue; }
                    log[s].push_back({epoch, t, st.write});
                }
            // bank conflicts: a 128-bit access is served in phases of 8 lanes; 8 distinct 16-byte bank groups needed
            for (int i = 0; i < kE; ++i)
                for (int l0 = 0; l0 < P; l0 += 8) {
                    int cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                    for (int l = l0; l < l0 + 8 && l < P; ++l) {
                        const int c = ++cnt[slot(st.kind, l, i) & 7];
                        if (c > worst_conflict) worst_conflict = c;
                    }
                }
            if (st.sync_after) { sync_kind.push_back(st.sync_after); ++epoch; }
        }
    sync_kind.push_back(0);
    int hazards = 0, used = 0;
    for (const auto& a : log) {
        if (!a.empty()) ++used;
        for (size_t x = 0; x < a.size(); ++x)
            for (size_t y = x + 1; y < a.size(); ++y) {
                if (a[x].thread == a[y].thread || !(a[x].write || a[y].write)) continue;
                bool ordered = false;
                for (int e = a[x].epoch; e < a[y].epoch && !ordered; ++e)
                    ordered = sync_kind[e] == 2 || (sync_kind[e] == 1 && a[x].thread / 32 == a[y].thread / 32);
                if (!ordered) ++hazards;
            }
    }
    // the frequency map must be a bijection onto 0..N-1
    std::vector<char> seen(N, 0);
    int dup = 0;
    for (int t = 0; t < P; ++t)
        for (int e = 0; e < kE; ++e) {
            const int k = D::freq_index(t, e);
            if (k < 0 || k >= N || seen[k]) ++dup; else seen[k] = 1;
        }
    out[0] = worst_conflict; out[1] = hazards; out[2] = oob; out[3] = used; out[4] = D::XLEN; out[5] = dup;
    return 0;
}
}  // namespace frs

extern "C" int frs_selftest_dif_host(int n, int inverse, const float* in, float* out) {
    if (!in || !out) return FRS_EINVAL;
    const float2* i2 = reinterpret_cast<const float2*>(in);
    float2* o2 = reinterpret_cast<float2*>(out);
    switch (n) {
        case 256: return frs::emu_dif<256>(inverse, i2, o2);
        case 512: return frs::emu_dif<512>(inverse, i2, o2);
        case 1024: return frs::emu_dif<1024>(inverse, i2, o2);
        case 2048: return frs::emu_dif<2048>(inverse, i2, o2);
        case 4096: return frs::emu_dif<4096>(inverse, i2, o2);
        default: return FRS_EINVAL;
    }
}

extern "C" int frs_selftest_dif_exchange(int n, int* out) {
    if (!out) return FRS_EINVAL;
    switch (n) {
        case 256: return frs::dif_exchange_report<256>(out);
        case 512: return frs::dif_exchange_report<512>(out);
        case 1024: return frs::dif_exchange_report<1024>(out);
        case 2048: return frs::dif_exchange_report<2048>(out);
        case 4096: return frs::dif_exchange_report<4096>(out);
        default: return FRS_EINVAL;
    }
}

extern "C" int frs_selftest_fft_host(int n, int inverse, const float* in, float* out) {
    if (!in || !out) return FRS_EINVAL;
    const float2* i2 = reinterpret_cast<const float2*>(in);
    float2* o2 = reinterpret_cast<float2*>(out);
    switch (n) {
        case 16: return frs::emu<16>(inverse, i2, o2);
        case 32: return frs::emu<32>(inverse, i2, o2);
        case 64: return frs::emu<64>(inverse, i2, o2);
        case 128: return frs::emu<128>(inverse, i2, o2);
        case 256: return frs::emu<256>(inverse, i2, o2);
        case 512: return frs::emu<512>(inverse, i2, o2);
        case 1024: return frs::emu<1024>(inverse, i2, o2);
        case 2048: return frs::emu<2048>(inverse, i2, o2);
        case 4096: return frs::emu<4096>(inverse, i2, o2);
        default: return FRS_EINVAL;
    }
}

// Geometry of the TMA tensor copies (tmap.h) for rows of nf bins and columns of `rows` samples:
// out = {box_bins, bin_copies, box_pairs, col_copies, xbuf_len(nf) [16-byte slots], tma usable for rows (0/1)}
extern "C" int frs_selftest_tma_geometry(int nf, int rows, int* out) {
    if (!out || nf < 16 || rows < 32 || (nf & (nf - 1)) || (rows & (rows - 1))) return FRS_EINVAL;
    out[0] = frs::tma_box_bins(nf);
    out[1] = frs::tma_bin_copies(nf);
    out[2] = frs::tma_box_pairs(rows);
    out[3] = frs::tma_col_copies(rows);
    out[4] = frs::xbuf_len(nf);
    out[5] = frs::tma_rows_ok(nf) ? 1 : 0;
    return 0;
}
