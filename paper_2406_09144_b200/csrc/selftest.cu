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
