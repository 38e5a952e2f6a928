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

// ---- tensor-core measurement owed by north_star ("tensor cores only if a DFT-as-GEMM stage is MEASURED to beat the radix
// passes"): throughput of tcgen05.mma kind::tf32 at the shape a radix-16 DFT stage needs -- M = 128 positions per
// instruction, K = 8, N = 32 or 64 real outputs, operands in shared memory, accumulator in TMEM, one CTA per SM.
// A stage of one column pair is 256 positions x K = 96 (3-term TF32 split of a 32-real input: hi.hi + lo.hi + hi.lo,
// needed for the 1e-5 parity bar) x N = 64 (even- and odd-bin outputs) = 24 such instructions.
// compares the result with the 640 SM-cycles the packed-FP32 butterflies of the same stage take.
namespace frs {
__device__ __forceinline__ unsigned st_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned long long st_make_desc(unsigned addr, unsigned lbo, unsigned sbo) {
    unsigned long long d = 0;                                       // SWIZZLE_NONE, K-major (canonical 8 x 16-byte core matrices)
    d |= (unsigned long long)((addr >> 4) & 0x3FFF);
    d |= (unsigned long long)((lbo >> 4) & 0x3FFF) << 16;
    d |= (unsigned long long)((sbo >> 4) & 0x3FFF) << 32;
    d |= 1ull << 46;                                                // descriptor version of sm_100
    return d;
}
template <int N>
__global__ void __launch_bounds__(128, 1) tcgen05_stage_kernel(int iters, int nmma, long long* cyc) {
    __shared__ __align__(1024) float a_s[128 * 8 * 2];
    __shared__ __align__(1024) float b_s[64 * 8 * 2];
    __shared__ unsigned tmem_base;
    __shared__ __align__(8) unsigned long long bar;
    for (int i = threadIdx.x; i < 128 * 16; i += 128) a_s[i] = 0.001f * (i % 97);
    for (int i = threadIdx.x; i < 64 * 16; i += 128) b_s[i] = 0.002f * (i % 89);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(st_smem_u32(&bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (threadIdx.x < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" :: "r"(st_smem_u32(&tmem_base)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = tmem_base;
    // instruction descriptor: D = F32 (bit 4), A = B = TF32 (2 at bits 7 and 10), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
    const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(N >> 3) << 17) | ((unsigned)(128 >> 4) << 24);
    const unsigned long long da = st_make_desc(st_smem_u32(a_s), 128, 256), db = st_make_desc(st_smem_u32(b_s), 128, 256);
    unsigned parity = 0;
    if (threadIdx.x == 0) {
        const long long t0 = clock64();
        for (int it = 0; it < iters; ++it) {
            for (int j = 0; j < nmma; ++j) {
                const unsigned acc = j > 0;
                asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                             :: "r"(tmem), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(st_smem_u32(&bar)) : "memory");
            unsigned ok = 0, spins = 0;
            while (!ok) {
                asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                             : "=r"(ok) : "r"(st_smem_u32(&bar)), "r"(parity) : "memory");
                if (!ok && ++spins > (1u << 24)) __trap();
            }
            parity ^= 1u;
        }
        if (blockIdx.x == 0) *cyc = clock64() - t0;
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (threadIdx.x < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" :: "r"(tmem) : "memory");
}
}  // namespace frs

extern "C" int frs_selftest_tcgen05_stage(int n_out, int mmas_per_commit, int iters, double* clk_per_mma) {
    if (!clk_per_mma || (n_out != 32 && n_out != 64) || mmas_per_commit < 1 || iters < 1) return FRS_EINVAL;
    int ndev = 0, sms = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return FRS_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    long long* d = nullptr;
    if (cudaMalloc(reinterpret_cast<void**>(&d), sizeof(long long)) != cudaSuccess) return FRS_ECUDA;
    for (int pass = 0; pass < 2; ++pass) {                          // warm-up, then the timed launch
        const int it = pass ? iters : 4;
        if (n_out == 32) frs::tcgen05_stage_kernel<32><<<sms, 128>>>(it, mmas_per_commit, d);
        else frs::tcgen05_stage_kernel<64><<<sms, 128>>>(it, mmas_per_commit, d);
        if (cudaDeviceSynchronize() != cudaSuccess) { cudaFree(d); return FRS_ECUDA; }
    }
    long long h = 0;
    cudaMemcpy(&h, d, sizeof(h), cudaMemcpyDeviceToHost);
    cudaFree(d);
    *clk_per_mma = (double)h / iters / mmas_per_commit;
    return 0;
}
