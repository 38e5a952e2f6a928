// fft_core.cuh -- register-resident Stockham FFT shared by a group of P = N/16 threads.
//
// Each thread owns kE = 16 complex elements of an N-point transform in the CANONICAL
// distribution  reg e  <->  position p + e*P  (p = thread index inside the group).  A stage of
// radix R does 16/R butterflies per thread fully in registers; between stages the group
// exchanges through a padded shared-memory buffer: one float4 slot per position (the pair of transforms a
// thread carries), one slot of padding per 16 (xpad).  The scatters and gathers of the stages are free of bank
// conflicts; a phase of 8 lanes that straddles a padding step is not -- which is why the mirror reads Z[N - k] of
// rows_fwd (kernels.cuh), whose phases are offset by one position, go through a DENSE parking layout instead (in the
// padded one they conflicted 2-way in half of their phases: 7 % of that kernel's shared-memory wavefronts).
// Input and output are both in natural order in the canonical distribution, so forward -> pointwise -> inverse
// needs no reordering.
//
// The stage arithmetic is __host__ __device__: csrc/selftest.cu replays it thread by thread on
// the CPU so that the index maps and twiddle tables are tested without a GPU.
#pragma once
#include <cuda_runtime.h>

#define FRS_HD __host__ __device__ __forceinline__

namespace frs {

constexpr int kE = 16;
constexpr float kSqrtHalf = 0.70710678118654752440f;
constexpr float kC1 = 0.92387953251128675613f;   // cos(pi/8)
constexpr float kS1 = 0.38268343236508977173f;   // sin(pi/8)
// exp(-i pi e/16), e = 0..15: the step between the kE canonical slots of a thread in the table
// twist[n] = exp(-i pi n / N)  (n = p + e N/16)
FRS_HD constexpr float cos_pi16(int e) {
    constexpr float t[16] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                             0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f, 0.19509032201612826785f,
                             0.0f, -0.19509032201612826785f, -0.38268343236508977173f, -0.55557023301960222474f,
                             -0.70710678118654752440f, -0.83146961230254523708f, -0.92387953251128675613f, -0.98078528040323044913f};
    return t[e];
}
FRS_HD constexpr float sin_pi16(int e) {
    constexpr float t[16] = {0.0f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                             0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f, 0.98078528040323044913f,
                             1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                             0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f, 0.19509032201612826785f};
    return t[e];
}

FRS_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
FRS_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
FRS_HD float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
FRS_HD float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }
// a * w
FRS_HD float2 cmul(float2 a, float2 w) {
    return make_float2(fmaf(-a.y, w.y, a.x * w.x), fmaf(a.y, w.x, a.x * w.y));
}
// a * conj(w)
FRS_HD float2 cmulc(float2 a, float2 w) {
    return make_float2(fmaf(a.y, w.y, a.x * w.x), fmaf(a.y, w.x, -(a.x * w.y)));
}
// ---- packed pairs ---------------------------------------------------------------------------------
// A thread advances TWO transforms that share every twiddle.  Their samples travel as one C2: the real
// parts of both in one float2, the imaginary parts in another (lane .x = transform 0, .y = transform 1).
// On sm_100a every add / multiply / fma on such a float2 is ONE packed instruction (FADD2 / FMUL2 /
// FFMA2: two fp32 results per issue slot, a scalar twiddle broadcast to both lanes for free), which
// halves the issue slots of the butterflies; the host build (selftest.cu) runs the same code with
// plain float arithmetic.
struct C2 { float2 re, im; };

FRS_HD float2 f2bc(float s) { return make_float2(s, s); }
FRS_HD float2 f2neg(float2 a) { return make_float2(-a.x, -a.y); }
FRS_HD float2 f2add(float2 a, float2 b) {
#ifdef __CUDA_ARCH__
    return __fadd2_rn(a, b);
#else
    return make_float2(a.x + b.x, a.y + b.y);
#endif
}
FRS_HD float2 f2sub(float2 a, float2 b) { return f2add(a, f2neg(b)); }
FRS_HD float2 f2mul(float2 a, float2 b) {
#ifdef __CUDA_ARCH__
    return __fmul2_rn(a, b);
#else
    return make_float2(a.x * b.x, a.y * b.y);
#endif
}
// a * b + c
FRS_HD float2 f2fma(float2 a, float2 b, float2 c) {
#ifdef __CUDA_ARCH__
    return __ffma2_rn(a, b, c);
#else
    return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y));
#endif
}
FRS_HD C2 c2zero() { C2 r; r.re = make_float2(0.f, 0.f); r.im = r.re; return r; }
FRS_HD C2 c2make(float2 a, float2 b) { C2 r; r.re = make_float2(a.x, b.x); r.im = make_float2(a.y, b.y); return r; }
FRS_HD float2 c2get(const C2& a, int t) { return t ? make_float2(a.re.y, a.im.y) : make_float2(a.re.x, a.im.x); }
FRS_HD C2 c2add(C2 a, C2 b) { C2 r; r.re = f2add(a.re, b.re); r.im = f2add(a.im, b.im); return r; }
FRS_HD C2 c2sub(C2 a, C2 b) { C2 r; r.re = f2sub(a.re, b.re); r.im = f2sub(a.im, b.im); return r; }
// both transforms times the same scalar complex w (forward) or conj(w) (inverse)
template <bool INV> FRS_HD C2 c2mul_dir(C2 a, float2 w) {
    C2 r;
    if (INV) {
        r.re = f2fma(a.im, f2bc(w.y), f2mul(a.re, f2bc(w.x)));
        r.im = f2fma(a.re, f2bc(-w.y), f2mul(a.im, f2bc(w.x)));
    } else {
        r.re = f2fma(a.im, f2bc(-w.y), f2mul(a.re, f2bc(w.x)));
        r.im = f2fma(a.re, f2bc(w.y), f2mul(a.im, f2bc(w.x)));
    }
    return r;
}
// a + s*(-i d) forward, a + s*(+i d) inverse, s = +1 (PLUS) or -1: the multiplication by -+i is only a
// choice of components and signs
template <bool INV, bool PLUS> FRS_HD C2 c2add_mi(C2 a, C2 d) {
    C2 r;
    if (INV != PLUS) { r.re = f2add(a.re, d.im); r.im = f2sub(a.im, d.re); }   // a + (d.im, -d.re)
    else             { r.re = f2sub(a.re, d.im); r.im = f2add(a.im, d.re); }   // a + (-d.im, d.re)
    return r;
}
// a * w8^K (forward w8 = exp(-2 pi i/8)); inverse uses the conjugate
template <int K, bool INV> FRS_HD C2 c2mul_w8(C2 a) {
    C2 r;
    if (K == 0) return a;
    if (K == 2) {
        if (INV) { r.re = f2neg(a.im); r.im = a.re; } else { r.re = a.im; r.im = f2neg(a.re); }
        return r;
    }
    const float2 h = f2bc(kSqrtHalf), mh = f2bc(-kSqrtHalf);
    if (K == 1) {
        if (INV) { r.re = f2mul(f2sub(a.re, a.im), h); r.im = f2mul(f2add(a.re, a.im), h); }
        else     { r.re = f2mul(f2add(a.re, a.im), h); r.im = f2mul(f2sub(a.im, a.re), h); }
    } else { /* K == 3 */
        if (INV) { r.re = f2mul(f2add(a.re, a.im), mh); r.im = f2mul(f2sub(a.re, a.im), h); }
        else     { r.re = f2mul(f2sub(a.im, a.re), h);  r.im = f2mul(f2add(a.re, a.im), mh); }
    }
    return r;
}
// a * w16^K, K in {0,1,2,3,4,6,9}
template <int K, bool INV> FRS_HD C2 c2mul_w16(C2 a) {
    if (K == 0) return a;
    if (K == 2) return c2mul_w8<1, INV>(a);
    if (K == 4) return c2mul_w8<2, INV>(a);
    if (K == 6) return c2mul_w8<3, INV>(a);
    const float2 w = (K == 1) ? make_float2(kC1, -kS1) : (K == 3) ? make_float2(kS1, -kC1) : make_float2(-kC1, kS1) /*K==9*/;
    return c2mul_dir<INV>(a, w);
}

// ---- small DFTs on packed pairs, natural order in and out, in place ----------------------------------
template <bool INV> FRS_HD void dft2(C2& a, C2& b) {
    const C2 t = a;
    a = c2add(t, b);
    b = c2sub(t, b);
}
template <bool INV> FRS_HD void dft4(C2& a0, C2& a1, C2& a2, C2& a3) {
    const C2 t0 = c2add(a0, a2), t1 = c2sub(a0, a2), t2 = c2add(a1, a3), d = c2sub(a1, a3);
    a0 = c2add(t0, t2);
    a2 = c2sub(t0, t2);
    a1 = c2add_mi<INV, true>(t1, d);
    a3 = c2add_mi<INV, false>(t1, d);
}
template <bool INV> FRS_HD void dft8(C2 (&t)[8]) {
    dft4<INV>(t[0], t[2], t[4], t[6]);   // E[k] in t[0],t[2],t[4],t[6]
    dft4<INV>(t[1], t[3], t[5], t[7]);   // O[k] in t[1],t[3],t[5],t[7]
    const C2 o0 = t[1], o1 = c2mul_w8<1, INV>(t[3]), o3 = c2mul_w8<3, INV>(t[7]), d2 = t[5];
    const C2 e0 = t[0], e1 = t[2], e2 = t[4], e3 = t[6];
    t[0] = c2add(e0, o0); t[4] = c2sub(e0, o0);
    t[1] = c2add(e1, o1); t[5] = c2sub(e1, o1);
    t[2] = c2add_mi<INV, true>(e2, d2); t[6] = c2add_mi<INV, false>(e2, d2);
    t[3] = c2add(e3, o3); t[7] = c2sub(e3, o3);
}
template <bool INV> FRS_HD void dft16(C2 (&t)[16]) {
    // n = 4 n1 + n0, k = k0 + 4 k1:  X[k] = sum_n0 w4^{n0 k1} w16^{n0 k0} sum_n1 w4^{n1 k0} a[4 n1 + n0]
    dft4<INV>(t[0], t[4], t[8], t[12]);      // n0 = 0: B[0][k0] at t[4 k0 + 0]
    dft4<INV>(t[1], t[5], t[9], t[13]);
    dft4<INV>(t[2], t[6], t[10], t[14]);
    dft4<INV>(t[3], t[7], t[11], t[15]);
    t[5] = c2mul_w16<1, INV>(t[5]);   t[6] = c2mul_w16<2, INV>(t[6]);   t[7] = c2mul_w16<3, INV>(t[7]);
    t[9] = c2mul_w16<2, INV>(t[9]);   t[10] = c2mul_w16<4, INV>(t[10]); t[11] = c2mul_w16<6, INV>(t[11]);
    t[13] = c2mul_w16<3, INV>(t[13]); t[14] = c2mul_w16<6, INV>(t[14]); t[15] = c2mul_w16<9, INV>(t[15]);
    dft4<INV>(t[0], t[1], t[2], t[3]);       // k0 = 0: X[0 + 4 k1] at t[k1]
    dft4<INV>(t[4], t[5], t[6], t[7]);       // k0 = 1: X[1 + 4 k1] at t[4 + k1]
    dft4<INV>(t[8], t[9], t[10], t[11]);
    dft4<INV>(t[12], t[13], t[14], t[15]);
    // transpose 4x4: X[k0 + 4 k1] currently at t[4 k0 + k1]
    C2 s;
    s = t[1]; t[1] = t[4]; t[4] = s;
    s = t[2]; t[2] = t[8]; t[8] = s;
    s = t[3]; t[3] = t[12]; t[12] = s;
    s = t[6]; t[6] = t[9]; t[9] = s;
    s = t[7]; t[7] = t[13]; t[13] = s;
    s = t[11]; t[11] = t[14]; t[14] = s;
}
template <int R, bool INV> struct Dft;
template <bool INV> struct Dft<2, INV> { static FRS_HD void run(C2 (&t)[2]) { dft2<INV>(t[0], t[1]); } };
template <bool INV> struct Dft<4, INV> { static FRS_HD void run(C2 (&t)[4]) { dft4<INV>(t[0], t[1], t[2], t[3]); } };
template <bool INV> struct Dft<8, INV> { static FRS_HD void run(C2 (&t)[8]) { dft8<INV>(t); } };
template <bool INV> struct Dft<16, INV> { static FRS_HD void run(C2 (&t)[16]) { dft16<INV>(t); } };

// ---- plan: radices per transform length ------------------------------------------------------
// 16:[16] 32:[16,2] 64:[8,8] 128:[16,8] 256:[16,16] 512:[8,8,8] 1024:[16,8,8] 2048:[16,16,8] 4096:[16,16,16]
FRS_HD constexpr int plan_stages(int n) { return n == 16 ? 1 : (n <= 256 ? 2 : 3); }
FRS_HD constexpr int plan_radix(int n, int s) {
    return n == 16   ? 16
         : n == 32   ? (s == 0 ? 16 : 2)
         : n == 64   ? 8
         : n == 128  ? (s == 0 ? 16 : 8)
         : n == 256  ? 16
         : n == 512  ? 8
         : n == 1024 ? (s == 0 ? 16 : 8)
         : n == 2048 ? (s <= 1 ? 16 : 8)
                     : 16;
}
FRS_HD constexpr int plan_ns(int n, int s) {   // product of the radices before stage s
    return s == 0 ? 1 : plan_ns(n, s - 1) * plan_radix(n, s - 1);
}
// ---- twiddle tables (shared memory, a few KB for any N) -----------------------------------------
// Stage s > 0, butterfly b, output r >= 1 needs w_r = exp(-2 pi i j r / (NS R)), j = (p + b P) mod NS.
//   NS <= 16: direct table of float4 D[q][j] = (w_{2q+1}, w_{2q+2}), q < R/2.
//   NS  > 16: only w_1 is tabulated, factorised over j = 16 a + c:  w_1 = A[a] C[c] (float2 each,
//             A[a] = exp(-2 pi i 16 a / (NS R)), C[c] = exp(-2 pi i c / (NS R))); w_2..w_{R-1} follow by a
//             product tree of depth <= 4 (squares and one multiply), which costs the same arithmetic
//             as applying a factorised table and far fewer shared-memory reads.
FRS_HD constexpr bool plan_tw_fact(int n, int s) { return plan_ns(n, s) > 16; }
FRS_HD constexpr int plan_tw_wa(int n, int s) { return plan_tw_fact(n, s) ? plan_ns(n, s) / 16 : plan_ns(n, s); }
FRS_HD constexpr int plan_tw_size(int n, int s) {      // float4 slots of stage s
    return s == 0 ? 0 : (plan_tw_fact(n, s) ? (plan_tw_wa(n, s) + 16) / 2 : (plan_radix(n, s) / 2) * plan_tw_wa(n, s));
}
FRS_HD constexpr int plan_tw_off(int n, int s) { return s <= 1 ? 0 : plan_tw_off(n, s - 1) + plan_tw_size(n, s - 1); }
FRS_HD constexpr int plan_tw_total(int n) {            // >= 1 so that allocations are non-empty
    return plan_tw_off(n, plan_stages(n) - 1) + plan_tw_size(n, plan_stages(n) - 1) + 1;
}
FRS_HD float2 csq(float2 a) { return make_float2(fmaf(a.x, a.x, -(a.y * a.y)), 2.0f * a.x * a.y); }
// w[r] = w[1]^r for r = 2..R-1
template <int R> FRS_HD void twiddle_powers(float2 (&w)[R]) {
    if (R > 2) { w[2] = csq(w[1]); w[3] = cmul(w[2], w[1]); }
    if (R > 4) { w[4] = csq(w[2]); w[5] = cmul(w[4], w[1]); w[6] = csq(w[3]); w[7] = cmul(w[4], w[3]); }
    if (R > 8) {
        w[8] = csq(w[4]);  w[9] = cmul(w[8], w[1]);  w[10] = csq(w[5]); w[11] = cmul(w[8], w[3]);
        w[12] = csq(w[6]); w[13] = cmul(w[8], w[5]); w[14] = csq(w[7]); w[15] = cmul(w[8], w[7]);
    }
}

FRS_HD constexpr int xpad(int pos) { return pos + (pos >> 4); }
// slots of one exchange buffer (holds positions 0..N inclusive: the row passes park X[N] too)
FRS_HD constexpr int xbuf_len(int n) { return (n + (n >> 4) + 8 + 7) & ~7; }   // multiple of 128 bytes (TMA boxes)

// exchange slot of one position: (re of transform 0, re of 1, im of 0, im of 1) -> 128-bit accesses
FRS_HD float4 pack(const C2& a) { return make_float4(a.re.x, a.re.y, a.im.x, a.im.y); }
FRS_HD C2 unpack(float4 s) { C2 r; r.re = make_float2(s.x, s.y); r.im = make_float2(s.z, s.w); return r; }

// ---- one stage: twiddle the inputs, butterfly, leave result r of butterfly b in v[b + r*NB] ----
// Both transforms of the pair are advanced by the same packed instructions.  tw: packed tables.
template <int N, int S, bool INV>
FRS_HD void stage_compute(C2 (&v)[kE], int p, const float4* __restrict__ tw) {
    constexpr int R = plan_radix(N, S), NB = kE / R, HP = R / 2, P = N / kE, NS = plan_ns(N, S);
    constexpr int WA = plan_tw_wa(N, S);
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        float2 w[R];
        if (S > 0) {
            const int j = (p + b * P) & (NS - 1);
            const float4* ta = tw + plan_tw_off(N, S);
            if (plan_tw_fact(N, S)) {
                const float2* fa = reinterpret_cast<const float2*>(ta);
                w[1] = cmul(fa[j >> 4], fa[WA + (j & 15)]);
                twiddle_powers<R>(w);
            } else {
#pragma unroll
                for (int q = 0; q < HP; ++q) {
                    const float4 ww = ta[q * WA + j];
                    w[2 * q + 1] = make_float2(ww.x, ww.y);
                    if (2 * q + 2 < R) w[2 * q + 2] = make_float2(ww.z, ww.w);
                }
            }
        }
        C2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = v[b + r * NB];
        if (S > 0) {
#pragma unroll
            for (int r = 1; r < R; ++r) x[r] = c2mul_dir<INV>(x[r], w[r]);
        }
        Dft<R, INV>::run(x);
#pragma unroll
        for (int r = 0; r < R; ++r) v[b + r * NB] = x[r];
    }
}
// Stockham position of output r of butterfly b of stage S
template <int N, int S>
FRS_HD int stage_pos(int p, int b, int r) {
    constexpr int R = plan_radix(N, S), P = N / kE, NS = plan_ns(N, S);
    const int j = p + b * P;
    return (j / NS) * NS * R + (j % NS) + r * NS;
}
template <int N, int S>
FRS_HD void stage_scatter2(const C2 (&v)[kE], int p, float4* buf) {
    constexpr int R = plan_radix(N, S), NB = kE / R;
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int r = 0; r < R; ++r) buf[xpad(stage_pos<N, S>(p, b, r))] = pack(v[b + r * NB]);
}
template <int N>
FRS_HD void canon_gather2(C2 (&v)[kE], int p, const float4* buf) {
    constexpr int P = N / kE;
#pragma unroll
    for (int e = 0; e < kE; ++e) v[e] = unpack(buf[xpad(p + e * P)]);
}
template <int N>
FRS_HD void canon_scatter2(const C2 (&v)[kE], int p, float4* buf) {
    constexpr int P = N / kE;
#pragma unroll
    for (int e = 0; e < kE; ++e) buf[xpad(p + e * P)] = pack(v[e]);
}

#ifdef __CUDACC__
// ---- group barrier -----------------------------------------------------------------------------------
// The P threads that share a transform synchronise on their own named barrier, so that the groups of
// a CTA drift apart freely: while one group exchanges through shared memory the other computes
// (measured on B200: butterflies and LDS/STS traffic of two groups of ONE CTA overlap, those of two
// co-resident CTAs hardly do).  Groups narrower than a warp fall back to the CTA-wide barrier 0.
struct GroupBar {
    int id, n;
    __device__ __forceinline__ void sync() const { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(n) : "memory"); }
};
// ---- the whole transform of a PAIR of sequences sharing twiddles ---------------------------------
// All threads of the group must call this.  buf: one exchange buffer of xbuf_len(N) float4, private
// to the group.  tw: packed twiddle table (shared memory).
template <int N, bool INV, int S>
__device__ __forceinline__ void pair_fft_from(C2 (&v)[kE], int p, float4* buf, const float4* __restrict__ tw, const GroupBar& gb) {
    if constexpr (S < plan_stages(N)) {
        stage_compute<N, S, INV>(v, p, tw);
        if constexpr (S + 1 < plan_stages(N)) {
            stage_scatter2<N, S>(v, p, buf);
            gb.sync();
            canon_gather2<N>(v, p, buf);
            gb.sync();
        }
        pair_fft_from<N, INV, S + 1>(v, p, buf, tw, gb);
    }
}
template <int N, bool INV>
__device__ __forceinline__ void pair_fft(C2 (&v)[kE], int p, float4* buf, const float4* __restrict__ tw, const GroupBar& gb) {
    pair_fft_from<N, INV, 0>(v, p, buf, tw, gb);
}
// The same transform in two halves, so that a caller can reuse `buf` (it is free after the head)
// while the last stage, which runs entirely in registers, is still to be computed.
template <int N, bool INV, int S>
__device__ __forceinline__ void pair_fft_head_from(C2 (&v)[kE], int p, float4* buf, const float4* __restrict__ tw, const GroupBar& gb) {
    if constexpr (S + 1 < plan_stages(N)) {
        stage_compute<N, S, INV>(v, p, tw);
        stage_scatter2<N, S>(v, p, buf);
        gb.sync();
        canon_gather2<N>(v, p, buf);
        gb.sync();
        pair_fft_head_from<N, INV, S + 1>(v, p, buf, tw, gb);
    }
}
template <int N, bool INV>
__device__ __forceinline__ void pair_fft_head(C2 (&v)[kE], int p, float4* buf, const float4* __restrict__ tw, const GroupBar& gb) {
    pair_fft_head_from<N, INV, 0>(v, p, buf, tw, gb);
}
template <int N, bool INV>
__device__ __forceinline__ void pair_fft_tail(C2 (&v)[kE], int p, const float4* __restrict__ tw) {
    stage_compute<N, plan_stages(N) - 1, INV>(v, p, tw);
}

// ---- asynchronous copies ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src_gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(void* dst_smem, const void* src_gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
// mbarrier + bulk (TMA) copy of a contiguous block global -> shared
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// the same block, only pulled into L2 (nothing to wait for)
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(src_gmem), "r"(bytes) : "memory");
}
// tensor (TMA) copies global -> shared of one box of a map, completion counted on an mbarrier
__device__ __forceinline__ void tensor_g2s_3d(void* dst_smem, const void* tmap, int c0, int c1, int c2, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 :: "r"(smem_u32(dst_smem)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tensor_g2s_4d(void* dst_smem, const void* tmap, int c0, int c1, int c2, int c3, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 :: "r"(smem_u32(dst_smem)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
// the same boxes, only pulled into L2 (no shared-memory destination, no completion to wait for)
__device__ __forceinline__ void tensor_prefetch_4d(const void* tmap, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
                 :: "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tensor_prefetch_5d(const void* tmap, int c0, int c1, int c2, int c3, int c4) {
    asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global.tile [%0, {%1, %2, %3, %4, %5}];"
                 :: "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tensor_g2s_5d(void* dst_smem, const void* tmap, int c0, int c1, int c2, int c3, int c4, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
                 :: "r"(smem_u32(dst_smem)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned ok, spins = 0;
    unsigned long long t0 = 0;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        // a copy that never completes (bad map, lost issue) must fail loudly, not hang the device: 2 s of wall time
        // on the global timer (a spin count would depend on clocks and on how long a try_wait suspends the warp)
        if (!ok && (++spins & 1023u) == 0) {
            unsigned long long t;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
            if (t0 == 0) t0 = t;
            else if (t - t0 > 2000000000ull) __trap();
        }
    } while (!ok);
}
// cooperative copy of the packed twiddle table into shared memory (all threads; caller syncs)
template <int N>
__device__ __forceinline__ void load_twiddles(float4* dst, const float4* __restrict__ src) {
    for (int i = threadIdx.x; i < plan_tw_total(N); i += blockDim.x) dst[i] = src[i];
}
#endif

}  // namespace frs
