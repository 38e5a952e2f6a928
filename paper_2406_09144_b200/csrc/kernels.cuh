// kernels.cuh -- the FFT passes of the fast-resolve hot path.
//
// Data layouts:
//   image      real  [nb][ny][nx]                      row-major, x fastest
//   spectrum T cplx  [nb][NF/8+1][ny/2][8][2]          128-byte blocks (8 bins kx) x (rows 2r, 2r+1), kx = 0..NF (the
//                                                       unused slots of the last block are never read):
//                                                       rows_fwd -> conv_cols (tmap.h)
//   spectrum T2 cplx [nb][2 ntile][ny]                 column kx contiguous: conv_cols -> rows_inv
//   weights Wt real  [nb][2 ntile (kx)][ny][2]         per column, (even-bin, odd-bin) weight pairs in the order the
//                                                       column pass consumes them (natural q for ny < 256, the
//                                                       permuted order of fft_dif.cuh otherwise)
//
// Passes (all persistent: a CTA walks work items blockIdx.x, blockIdx.x + gridDim.x, ...; the stage
// twiddles live in shared memory, loaded once per CTA):
//   rows_fwd   real rows -> half spectrum (R2C through a half-length complex FFT), PAD = the row
//              is zero-extended nx -> 2 nx (Eq. 14 'FFT[P I]'), optional fused multiply
//   conv_cols  per column: zero-padded FFT (even/odd split) . W . inverse FFT, cropped (Eq. 14)
//   rows_inv   half spectrum -> real rows, cropped to the first nx samples (P:182 'P^dagger'),
//              fused epilogues (x s, energy/residual)
//   hart_cols  second pass of the 2-D Hartley transform of the correlated field (reading R6)
// Every thread carries a PAIR of transforms (two rows / the two columns of a tile): they share the
// twiddle fetches and travel through shared memory as one float4 per position.
#pragma once
#include <type_traits>
#include "fft_core.cuh"
#include "fft_dif.cuh"
#include "tmap.h"

namespace frs {

// CTA geometry.  ROLES: thread groups of P cooperating on one work item (conv_cols: even/odd bins).
// STAGE: extra float4 slots per group for an asynchronously filled staging buffer.
template <int NF, int ROLES, int STAGE = 0, int BIG = 512>
struct Geo {
    static constexpr int P = NF / kE;                                  // threads per transform pair
    static constexpr int GT = P * ROLES;                               // threads per group
    // BIG = 512: one CTA per SM whose groups overlap each other's phases; 256: two CTAs per SM
    // (128 registers per thread either way) -- chosen per kernel by measurement
    static constexpr int WANT = NF >= 1024 ? BIG : (NF >= 256 ? 256 : 64);
    static constexpr int THREADS = GT >= WANT ? GT : WANT;
    static constexpr int G = THREADS / GT;                             // groups per CTA
    static constexpr bool OWN_BAR = (GT % 32 == 0) && G <= 15 && ROLES == 1;   // a named barrier per group
    static constexpr int TW = (plan_tw_total(NF) + 7) & ~7;            // float4 slots of the twiddle tables (128-byte multiple)
    static constexpr int GROUP_SLOTS = ROLES * xbuf_len(NF) + STAGE;   // float4 slots per group
    static constexpr int BAR_SLOTS = (G + 1) / 2;                      // one 8-byte mbarrier per group
    static constexpr int SMEM = (TW + G * GROUP_SLOTS + BAR_SLOTS) * (int)sizeof(float4);
    static constexpr int MINB = THREADS >= 512 ? 1 : (THREADS >= 256 ? 2 : 4);
    __device__ static GroupBar bar(int g) { return OWN_BAR ? GroupBar{1 + g, GT} : GroupBar{0, THREADS}; }
};

// Streaming data (images, spectrum tiles, weights) bypasses L1 allocation so that the twist
// tables, fetched with plain __ldg, stay L1-resident.  The read-only loads are NOT volatile and the
// stores carry no "memory" clobber: the compiler must be free to hoist a whole batch of loads above
// the arithmetic and stores of the previous element, otherwise every load-use-store triple pays the
// full memory latency in sequence.  (No kernel reads back what it stored.)
__device__ __forceinline__ float2 ldg2(const float* p) {
    float2 r;
    asm("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ldg4(const void* p) {
    float4 r;
    asm("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
        : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ float ldg1(const float* p) {
    float r;
    asm("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ void stg4(void* p, float4 v) {
    asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w));
}
__device__ __forceinline__ void stg2(void* p, float2 v) {
    asm volatile("st.global.L1::no_allocate.v2.f32 [%0], {%1, %2};" :: "l"(p), "f"(v.x), "f"(v.y));
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

template <int NF> struct RowsGeo : Geo<NF, 1, 0, 256> {};
// padded row pass: plus a staging buffer of 2 rows of NF floats per group (the next item's input lands there while this
// item's transform owns the exchange buffer)
template <int NF> struct RowsFwdGeo : Geo<NF, 1, NF / 2, 256> {};

// ------------------------------------------------------------------------------------------------
struct RowsFwdArgs {
    const float* in;      // [nb][ny][nxr]
    const float* mul;     // optional [nb][ny][nxr] multiplier (s or A); nullptr = none
    float2* out;          // [nb][NF/B+1][ny/2][B][2]: blocks of B bins x (rows 2r, 2r+1); B = 8 (PAD) or 2, tmap.h
    int ny;               // rows
    int items_per_batch, nitems;
    size_t in_bstride, mul_bstride;   // elements (float)
    float scale;
    const float4* tw;     // packed stage twiddles for NF (global; copied to shared memory)
    const float2* twist;  // exp(-2 pi i k/(2 NF)), k = 0..NF
};

// One group (P threads) transforms rows y0, y0+1 together.  Software pipeline (PAD): the two input rows of the NEXT item
// are pulled by one bulk TMA copy into a staging buffer of their own as soon as this item has picked its rows up, so the
// copy has a whole transform to land (when it landed in the exchange buffer it could only start behind the transform and
// 16 % of the warp time was spent waiting for it, profiles/r1_l1_apply_ncu.md); the rows of the multiplier are read
// straight into registers, from L2: a bulk prefetch pulls them in one item ahead.  Unpadded rows (Hartley pass) are
// twice as long and load directly.
// Unpacking X[k] from the half-length transform Z needs Z[k] (still in the thread's registers) and
// Z[NF-k] (another thread's): Z is parked in the exchange buffer once and every thread reads its 16
// mirror slots.  A thread then holds X[k] of both rows (16 bytes); neighbouring lanes hold
// neighbouring bins, so each lane pair stores one whole 32-byte sector of the block layout.
template <int NF, bool PAD>
__global__ void __launch_bounds__(RowsGeo<NF>::THREADS, RowsGeo<NF>::MINB)
rows_fwd_kernel(RowsFwdArgs a) {
    using GEO = typename std::conditional<PAD, RowsFwdGeo<NF>, RowsGeo<NF>>::type;
    constexpr int P = GEO::P;
    constexpr int NXR = PAD ? NF : 2 * NF;        // real samples per row
    constexpr int NE = PAD ? kE / 2 : kE;         // canonical slots that hold data
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    const GroupBar gb = GEO::bar(g);
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();

    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem4 + GEO::TW + (size_t)GEO::G * GEO::GROUP_SLOTS) + g;
    if (PAD && p == 0) mbar_init(bar, 1);
    unsigned parity = 0;
    const float* stg = reinterpret_cast<const float*>(buf + xbuf_len(NF));       // staged rows: x row 0, x row 1
    auto row_pair = [&](int item, int& b, int& rp) {
        b = item / a.items_per_batch;
        rp = (item - b * a.items_per_batch) * GEO::G + g;
        return item < a.nitems && 2 * rp < a.ny;
    };
    auto stage_rows = [&](int item) {                              // PAD only: 2 rows of NF floats; multiplier rows -> L2
        int b, rp;
        if (row_pair(item, b, rp) && p == 0) {
            fence_proxy_async();
            mbar_expect_tx(bar, 2 * NF * 4);
            bulk_g2s(const_cast<float*>(stg), a.in + b * a.in_bstride + (size_t)(2 * rp) * NXR, 2 * NF * 4, bar);
            if (a.mul) bulk_prefetch_l2(a.mul + b * a.mul_bstride + (size_t)(2 * rp) * NXR, 2 * NF * 4);
        }
        __syncwarp();   // the issuing lane must not be left behind a warp that spins on the mbarrier
    };
    // warm L2 with the rows of the item after this one (unpadded rows)
    auto prefetch_rows = [&](int item) {
        int b, rp;
        if (row_pair(item, b, rp)) {
            for (int i = p * 32; i < 2 * NXR; i += P * 32) {
                prefetch_l2(a.in + b * a.in_bstride + (size_t)(2 * rp) * NXR + i);
                if (a.mul) prefetch_l2(a.mul + b * a.mul_bstride + (size_t)(2 * rp) * NXR + i);
            }
        }
    };
    __syncthreads();
    if (PAD) stage_rows(blockIdx.x);

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        int b, rp;                                                 // batch, row pair
        const bool live = row_pair(item, b, rp);
        const int y0 = 2 * rp;
        float2 xin[2][NE], min_[2][NE];
#pragma unroll
        for (int e = 0; e < NE; ++e) { xin[0][e] = xin[1][e] = make_float2(0.f, 0.f); min_[0][e] = min_[1][e] = make_float2(1.f, 1.f); }
        if (live && a.mul) {
            const float* m0 = a.mul + b * a.mul_bstride + (size_t)y0 * NXR;
#pragma unroll
            for (int e = 0; e < NE; ++e) {
                min_[0][e] = ldg2(m0 + 2 * (p + e * P));
                min_[1][e] = ldg2(m0 + NXR + 2 * (p + e * P));
            }
        }
        if (PAD) {
            if (live) {
                mbar_wait(bar, parity);
                parity ^= 1u;
#pragma unroll
                for (int e = 0; e < NE; ++e) {
#pragma unroll
                    for (int t = 0; t < 2; ++t) xin[t][e] = *reinterpret_cast<const float2*>(stg + t * NF + 2 * (p + e * P));
                }
            }
            // the staged rows have been read (and the mirror slots of the previous item: the exchange buffer is free)
            gb.sync();
            stage_rows(item + gridDim.x);
        } else {
            if (live) {
                const float* r0 = a.in + b * a.in_bstride + (size_t)y0 * NXR;
#pragma unroll
                for (int e = 0; e < NE; ++e) {
                    xin[0][e] = ldg2(r0 + 2 * (p + e * P));
                    xin[1][e] = ldg2(r0 + NXR + 2 * (p + e * P));
                }
            }
            prefetch_rows(item + gridDim.x);
        }

        C2 v[kE];
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            if (e < NE) {
                float2 x[2];
#pragma unroll
                for (int t = 0; t < 2; ++t) x[t] = make_float2(xin[t][e].x * min_[t][e].x, xin[t][e].y * min_[t][e].y);
                v[e] = c2make(x[0], x[1]);
            } else {
                v[e] = c2zero();
            }
        }
        pair_fft<NF, false>(v, p, buf, tws, gb);
        // park Z DENSELY: slot k = (Z_0[k], Z_1[k]).  The mirror reads below walk the slots downwards in phases of 8 lanes that
        // are offset by one position; in the padded layout of the exchanges such a phase straddles a padding step and
        // conflicts 2-way (7 % of this kernel's shared-memory wavefronts, profiles/); any 8 consecutive dense slots do not
#pragma unroll
        for (int e = 0; e < kE; ++e) buf[p + e * P] = pack(v[e]);
        gb.sync();
        // X[k] scale = (Z[k] + conj Z[NF-k]) - i twist[k] (Z[k] - conj Z[NF-k]),  k = p + e P (and k = NF from Z[0])
        C2 xn = c2zero();
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int k = p + e * P;
            const C2 zm = unpack(buf[(NF - k) & (NF - 1)]);
            const float2 w0 = __ldg(a.twist + k);
            const float2 w = make_float2(w0.x * a.scale, w0.y * a.scale);     // the output scale rides on the twist ...
            const float2 sc = f2bc(a.scale);                                  // ... and on one fma per component
            C2 s, d0;
            s.re = f2add(v[e].re, zm.re);  s.im = f2sub(v[e].im, zm.im);
            d0.re = f2sub(v[e].re, zm.re); d0.im = f2add(v[e].im, zm.im);
            const C2 d = c2mul_dir<false>(d0, w);
            if (e == 0 && p == 0) {               // k = 0: twist[NF] = -1 gives X[NF] from the same Z[0]
                xn.re = f2fma(s.re, sc, f2neg(d.im));
                xn.im = f2fma(s.im, sc, d.re);
            }
            v[e].re = f2fma(s.re, sc, d.im);
            v[e].im = f2fma(s.im, sc, f2neg(d.re));
        }
        if (!PAD) gb.sync();                      // every mirror slot has been read (PAD: the barrier at the top of the next item)
        if (live) {
            // (X_0[k], X_1[k]) -> 16-byte slot k % 8 of block (k / 8, y0 / 2): 8 neighbouring lanes fill one 128-byte line
            auto slot = [](const C2& x) { return make_float4(x.re.x, x.im.x, x.re.y, x.im.y); };
            constexpr int BINS = PAD ? kBlockBins : kPairBins;    // tmap.h: 128-byte blocks for the convolution, pairs otherwise
            float4* ob = reinterpret_cast<float4*>(a.out + b * spec_batch_stride(a.ny, NF, BINS));
#pragma unroll
            for (int e = 0; e < kE; ++e) stg4(ob + spec_index(a.ny, p + e * P, y0, BINS) / 2, slot(v[e]));
            if (p == 0) stg4(ob + spec_index(a.ny, NF, y0, BINS) / 2, slot(xn));
        }
    }
}

#include "kernels_cols.inl"
#include "kernels_cols_dif.inl"
#include "kernels_inv.inl"
#include "kernels_inv_hart.inl"

}  // namespace frs
