// fft_dif.cuh -- second FFT core: forward transform decimated in frequency, inverse decimated in time,
// for the column convolution (forward -> pointwise weights -> inverse), N = 256 .. 4096.
//
// The spectrum between the two transforms may be in ANY order (the weights are stored in the order the
// threads consume them), so nothing has to be sorted.  That allows an exchange pattern in which
//   * every thread overwrites exactly the shared-memory slots it has just read itself (no write-after-read
//     hazard anywhere, hence no "buffer free" barrier),
//   * one of the two exchanges of a transform stays inside a group of C <= 16 neighbouring lanes
//     (__syncwarp instead of a block barrier: the warps of a group drift apart and overlap each other's
//     shared-memory and arithmetic phases),
//   * every address is one per-thread base plus a compile-time offset, and every access is free of bank
//     conflicts (checked lane by lane on the CPU: frs_selftest_dif_exchange, tests/test_host_logic.py).
// A forward + inverse pair costs TWO block barriers where the sorting (Stockham) core needs eight.
//
// Index algebra.  N = 256 C (C = 1, 2, 4, 8, 16), P = N/16 = 16 C threads, 16 elements per thread.
//   time       n = n0 + C n1 + P n2        n0 < C, n1 < 16, n2 < 16        (p = n0 + C n1 is the thread)
//   frequency  k = k0 + 16 k1 + 256 k2     k0 < 16, k1 < 16, k2 < C
//   w_N^{nk} = w_16^{n2 k0} . w_N^{p k0} . w_16^{n1 k1} . w_{16C}^{n0 k1} . w_C^{n0 k2}
//            =   stage A    .   tw1      .   stage B    .     tw2         .  stage C
// Roles of a thread t (same t, three decodings), registers v[0..15]:
//   time role   t = p;                v[n2]  /  after stage A: v[k0]
//   mid  role   t <-> (n0, k0);       v[n1]  /  after stage B: v[k1]
//   freq role   t <-> (j,  k0);       v[r NBC + b], r = n0 (then k2), k1 = j + C b, NBC = 16 / C
// Exchange buffer X: one region of RP slots (float4: the pair of transforms a thread carries) per k0;
// slot(k0, n0 + C t1) = RP k0 + n0 + CP t1  with t1 = n1 or k1 (CP = C + pad).
//   X1 (block-wide):  time role writes slot(k0 = i, p), i = 0..15;  mid role reads slot(k0, n0 + C i)
//   X2 (C lanes):     mid role writes slot(k0, n0 + C i) (the slots it read);  freq role reads
//                     slot(k0, r + C (j + C b))
// and the inverse runs the same four accesses backwards, again writing where the thread last read.
#pragma once
#include "fft_core.cuh"

namespace frs {

template <int N>
struct Dif {
    static_assert(N >= 256 && N <= 4096 && (N & (N - 1)) == 0, "Dif core: 256 <= N <= 4096");
    static constexpr int C = N / 256;
    static constexpr int P = N / kE;
    static constexpr int NBC = kE / C;
    static constexpr int CP = C >= 8 ? C + 1 : C;                   // slots per run of C positions
    static constexpr int RP = C >= 8 ? 16 * CP : 16 * C + 1;        // slots per k0 region
    static constexpr int XLEN = (16 * RP + 7) & ~7;                 // slots of the exchange buffer (128-byte multiple)
    static constexpr int KW = C >= 8 ? 1 : (P < 32 ? P : 32) / C;   // k0 values interleaved in a warp (C <= 4)
    // twiddle table (float4 slots): D[q C + n0] = (w^(2q+1), w^(2q+2)), w = w_{16C}^{n0}, q < 8   (tw2, direct)
    //                               then float2 TA[a] = w_N^{16 a} (a < C), TC[c] = w_N^c (c < 16)  (tw1, factorised)
    static constexpr int TW_D = C > 1 ? 8 * C : 0;
    static constexpr int TW_TOTAL = (TW_D + (C + 16 + 1) / 2 + 7) & ~7;

    // (n0, k0) of thread t in the mid role; (j, k0) in the freq role
    FRS_HD static int mid_n0(int t) { return C >= 8 ? t % C : (t % 32) / KW; }
    FRS_HD static int mid_k0(int t) { return C >= 8 ? t / C : (t % KW) + KW * (t / 32); }
    FRS_HD static int base_time(int t) { return (t % C) + CP * (t / C); }
    FRS_HD static int base_mid(int t) { return RP * mid_k0(t) + mid_n0(t); }
    FRS_HD static int base_freq(int t) { return RP * mid_k0(t) + CP * mid_n0(t); }
    FRS_HD static constexpr int off_time(int i) { return RP * i; }
    FRS_HD static constexpr int off_mid(int i) { return CP * i; }
    FRS_HD static constexpr int off_freq(int e) { return (e / NBC) + CP * C * (e % NBC); }   // e = r NBC + b
    // frequency index held by register e of thread t after the forward transform
    FRS_HD static int freq_index(int t, int e) { return mid_k0(t) + 16 * (mid_n0(t) + C * (e % NBC)) + 256 * (e / NBC); }
};

// ---- the four accesses -------------------------------------------------------------------------
template <int N> FRS_HD void dif_put_time(const C2 (&v)[kE], int t, float4* X) {
    float4* b = X + Dif<N>::base_time(t);
#pragma unroll
    for (int i = 0; i < kE; ++i) b[Dif<N>::off_time(i)] = pack(v[i]);
}
template <int N> FRS_HD void dif_get_time(C2 (&v)[kE], int t, const float4* X) {
    const float4* b = X + Dif<N>::base_time(t);
#pragma unroll
    for (int i = 0; i < kE; ++i) v[i] = unpack(b[Dif<N>::off_time(i)]);
}
template <int N> FRS_HD void dif_put_mid(const C2 (&v)[kE], int t, float4* X) {
    float4* b = X + Dif<N>::base_mid(t);
#pragma unroll
    for (int i = 0; i < kE; ++i) b[Dif<N>::off_mid(i)] = pack(v[i]);
}
template <int N> FRS_HD void dif_get_mid(C2 (&v)[kE], int t, const float4* X) {
    const float4* b = X + Dif<N>::base_mid(t);
#pragma unroll
    for (int i = 0; i < kE; ++i) v[i] = unpack(b[Dif<N>::off_mid(i)]);
}
template <int N> FRS_HD void dif_put_freq(const C2 (&v)[kE], int t, float4* X) {
    float4* b = X + Dif<N>::base_freq(t);
#pragma unroll
    for (int e = 0; e < kE; ++e) b[Dif<N>::off_freq(e)] = pack(v[e]);
}
template <int N> FRS_HD void dif_get_freq(C2 (&v)[kE], int t, const float4* X) {
    const float4* b = X + Dif<N>::base_freq(t);
#pragma unroll
    for (int e = 0; e < kE; ++e) v[e] = unpack(b[Dif<N>::off_freq(e)]);
}

// ---- twiddles -----------------------------------------------------------------------------------
// tw1: v[k0] *= w_N^{p k0} (conjugated for the inverse), the powers from one factorised base by the product tree
template <int N, bool INV> FRS_HD void dif_tw1(C2 (&v)[kE], int t, const float4* __restrict__ tw) {
    const float2* f = reinterpret_cast<const float2*>(tw + Dif<N>::TW_D);
    float2 w[kE];
    w[1] = cmul(f[t >> 4], f[Dif<N>::C + (t & 15)]);
    twiddle_powers<kE>(w);
#pragma unroll
    for (int k = 1; k < kE; ++k) v[k] = c2mul_dir<INV>(v[k], w[k]);
}
// tw2: v[k1] *= w_{16C}^{n0 k1}, direct table
template <int N, bool INV> FRS_HD void dif_tw2(C2 (&v)[kE], int t, const float4* __restrict__ tw) {
    if (Dif<N>::C == 1) return;
    const float4* d = tw + Dif<N>::mid_n0(t);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float4 ww = d[q * Dif<N>::C];
        v[2 * q + 1] = c2mul_dir<INV>(v[2 * q + 1], make_float2(ww.x, ww.y));
        if (2 * q + 2 < kE) v[2 * q + 2] = c2mul_dir<INV>(v[2 * q + 2], make_float2(ww.z, ww.w));
    }
}
// stage C: NBC butterflies of radix C over r, v[r NBC + b]
template <int N, bool INV> FRS_HD void dif_stage_c(C2 (&v)[kE]) {
    constexpr int C = Dif<N>::C, NBC = Dif<N>::NBC;
    if constexpr (C > 1) {
#pragma unroll
        for (int b = 0; b < NBC; ++b) {
            C2 x[C];
#pragma unroll
            for (int r = 0; r < C; ++r) x[r] = v[r * NBC + b];
            Dft<C, INV>::run(x);
#pragma unroll
            for (int r = 0; r < C; ++r) v[r * NBC + b] = x[r];
        }
    }
}

// ---- the transforms in phases (a phase = what a thread does between two synchronisations), so that
// the kernels can interleave their own work and the CPU replay can run them thread by thread ----------
// forward:  F0 | block barrier | F1 | warp sync | F2        (time role in, freq role out)
template <int N> FRS_HD void dif_fwd_0(C2 (&v)[kE], int t, float4* X, const float4* __restrict__ tw) {
    dft16<false>(v);
    dif_tw1<N, false>(v, t, tw);
    dif_put_time<N>(v, t, X);
}
template <int N> FRS_HD void dif_fwd_1(C2 (&v)[kE], int t, float4* X, const float4* __restrict__ tw) {
    dif_get_mid<N>(v, t, X);
    dft16<false>(v);
    if (Dif<N>::C > 1) {
        dif_tw2<N, false>(v, t, tw);
        dif_put_mid<N>(v, t, X);
    }
}
template <int N> FRS_HD void dif_fwd_2(C2 (&v)[kE], int t, const float4* X) {
    if (Dif<N>::C > 1) {
        dif_get_freq<N>(v, t, X);
        dif_stage_c<N, false>(v);
    }
}
// inverse:  I0 | warp sync | I1 | block barrier | I2        (freq role in, time role out)
template <int N> FRS_HD void dif_inv_0(C2 (&v)[kE], int t, float4* X) {
    if (Dif<N>::C > 1) {
        dif_stage_c<N, true>(v);
        dif_put_freq<N>(v, t, X);
    }
}
template <int N> FRS_HD void dif_inv_1(C2 (&v)[kE], int t, float4* X, const float4* __restrict__ tw) {
    if (Dif<N>::C > 1) {
        dif_get_mid<N>(v, t, X);
        dif_tw2<N, true>(v, t, tw);
    }
    dft16<true>(v);
    dif_put_mid<N>(v, t, X);
}
template <int N> FRS_HD void dif_inv_2(C2 (&v)[kE], int t, const float4* X, const float4* __restrict__ tw) {
    dif_get_time<N>(v, t, X);
    dif_tw1<N, true>(v, t, tw);
    dft16<true>(v);
}

#ifdef __CUDACC__
template <int N>
__device__ __forceinline__ void dif_load_twiddles(float4* dst, const float4* __restrict__ src) {
    for (int i = threadIdx.x; i < Dif<N>::TW_TOTAL; i += blockDim.x) dst[i] = src[i];
}
// the C lanes that share k0 are neighbours inside one warp
__device__ __forceinline__ void dif_warp_sync() { __syncwarp(); }
#endif

}  // namespace frs
