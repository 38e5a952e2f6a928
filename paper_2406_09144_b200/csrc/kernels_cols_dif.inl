// kernels_cols_dif.inl -- column convolution on the DIF/DIT core (included inside namespace frs by kernels.cuh)
//
// Same operation and the same staging scheme as conv_cols_kernel (kernels_cols.inl), for NF >= 256, on the
// FFT core of fft_dif.cuh: the spectrum between the forward and the inverse transform stays in the permuted
// order of that core (the weights are stored in it, k_setup.cu weights_permute), every exchange overwrites the
// slots the thread has just read, and one exchange of each transform stays inside C neighbouring lanes.  Per
// column a group passes TWO blocking barriers (eight in the sorting core).  The staging buffer holds columns only
// (the next one is in flight for a whole column time); the weights come from L2 straight into registers.
//
// Attribution builds (profiles/r3_conv_cols_attribution.md): compiling with -DFRS_STRIP=<mask> removes ingredients of this
// kernel so that the time of what is left can be read; the results are then WRONG by construction (frs_version() says so and
// bench.py marks its line).  Bits: 1 output stores, 2 weight loads (constant weights), 4 column fetch and its wait (stale
// staging data), 8 staging reads, 16 the FFT stages (memory skeleton), 32 twist-table loads.  Default 0: the product kernel,
// token for token.
#ifndef FRS_STRIP
#define FRS_STRIP 0
#endif
constexpr bool kStripStore = (FRS_STRIP & 1) != 0, kStripWeights = (FRS_STRIP & 2) != 0, kStripFetch = (FRS_STRIP & 4) != 0,
               kStripStage = (FRS_STRIP & 8) != 0, kStripFft = (FRS_STRIP & 16) != 0, kStripTwist = (FRS_STRIP & 32) != 0;

template <int NF> struct ColsDifGeo {
    using D = Dif<NF>;
    static constexpr int P = D::P;
    static constexpr int WANT = NF >= 1024 ? 512 : 256;
    static constexpr int THREADS = P >= WANT ? P : WANT;
    static constexpr int G = THREADS / P;                               // groups (columns in flight) per CTA
    static constexpr bool OWN_BAR = (P % 32 == 0) && G <= 15;           // named barrier 1 + g per group (exchange)
    static constexpr int TW = D::TW_TOTAL;                              // float4 slots, multiple of 8
    static constexpr int STAGE = NF / 2;                                // float4 slots of the staging buffer (NF float2)
    static constexpr int GROUP_SLOTS = D::XLEN + STAGE;
    static constexpr int BAR_SLOTS = (G + 1) / 2;
    static constexpr int SMEM = (TW + G * GROUP_SLOTS + BAR_SLOTS) * (int)sizeof(float4);
    static constexpr int MINB = THREADS >= 512 ? 1 : 2;
};

template <int NF>
__global__ void __launch_bounds__(ColsDifGeo<NF>::THREADS, ColsDifGeo<NF>::MINB)
conv_cols_dif_kernel(const __grid_constant__ ConvColsArgs a) {
    using GEO = ColsDifGeo<NF>;
    using D = Dif<NF>;
    constexpr int P = GEO::P;
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, t = threadIdx.x % P;
    float4* X = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    float2* stage = reinterpret_cast<float2*>(X + D::XLEN);                            // [NF] float2
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem4 + GEO::TW + (size_t)GEO::G * GEO::GROUP_SLOTS) + g;
    const GroupBar gb = GEO::OWN_BAR ? GroupBar{1 + g, P} : GroupBar{0, GEO::THREADS};
    dif_load_twiddles<NF>(tws, a.tw);
    if (t == 0) mbar_init(bar, 1);
    // twist^n for the thread's samples n = t + e P, from the exactly rounded table.  Only its first half is read
    // (twist^(NF-m) = -conj twist^m), so that it stays resident in the few KB of L1 this kernel leaves
    auto twist_e = [&](int e) {
        if (kStripTwist) return make_float2(0.6f + 1e-3f * (float)e, 0.8f);
        if (e < kE / 2) return __ldg(a.twist + t + e * P);
        const float2 c = __ldg(a.twist + (NF - e * P) - t);
        return make_float2(-c.x, c.y);
    };

    constexpr int BOXR = tma_box_pairs(NF), NCOPY = tma_col_copies(NF);
    auto column = [&](int item, bool& live, int& b, int& kx, const float*& w) {
        b = item / a.items_per_batch;
        kx = (item - b * a.items_per_batch) * GEO::G + g;
        live = item < a.nitems && kx < a.ncols;
        w = a.wt + b * a.w_bstride + (size_t)kx * NF * 2;
    };
    // this column's weights do not pass through shared memory: their 8 NF bytes are pulled into L2 one column ahead
    // (one bulk prefetch) and read from there straight into registers, so that the staging buffer belongs to the
    // columns alone and the NEXT column is in flight for a whole column time
    auto prefetch_weights = [&](const void* src, bool live) {
        if (t == 0 && live && !kStripWeights) bulk_prefetch_l2(src, NF * 8);
    };
    auto fetch_column = [&](int b, int kx, bool live) {          // column kx lands as NF contiguous samples
        if (kStripFetch) return;
        if (t == 0 && live) {
            fence_proxy_async();
            mbar_expect_tx(bar, NF * 8);
        }
        __syncwarp();
        if (t < NCOPY && live) tensor_g2s_5d(stage + 2 * BOXR * t, &a.tmap, 0, kx % kBlockBins, BOXR * t, kx / kBlockBins, b, bar);
        __syncwarp();
    };
    unsigned parity = 0;
    __syncthreads();
    {
        bool live; int b, kx; const float* w;
        column(blockIdx.x, live, b, kx, w);
        fetch_column(b, kx, live);
        prefetch_weights(w, live);
    }

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        bool live; int b, kx; const float* w;
        column(item, live, b, kx, w);

        C2 v[kE];
        if (live) {
            if (!kStripFetch) mbar_wait(bar, parity);
            parity ^= 1u;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 x = kStripStage ? make_float2(1e-3f * (float)(t + e), 1.0f - 1e-3f * (float)item) : stage[t + e * P];
                v[e] = c2make(x, cmul(x, twist_e(e)));                 // even bins: x, odd bins: x twist^n
            }
        } else {
#pragma unroll
            for (int e = 0; e < kE; ++e) v[e] = c2zero();
        }
        if (!kStripFft) dif_fwd_0<NF>(v, t, X, tws);
        gb.sync();                                  // X1 written; and every thread has picked up its samples:
        {                                           // the next column may land
            bool nlive; int nb_, nkx; const float* nw;
            column(item + gridDim.x, nlive, nb_, nkx, nw);
            fetch_column(nb_, nkx, nlive);
            prefetch_weights(nw, nlive);
        }
        if (!kStripFft) {
            dif_fwd_1<NF>(v, t, X, tws);
            dif_warp_sync();
            dif_fwd_2<NF>(v, t, X);
        }
        if (live) {
            const float* wp = w + 2 * t;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 ww = kStripWeights ? make_float2(1.0001f, 0.9999f - 1e-4f * (float)e)
                                                : ldg2(wp + 2 * e * P);   // (even-bin weight, odd-bin weight) of register e
                v[e].re = f2mul(v[e].re, ww);
                v[e].im = f2mul(v[e].im, ww);
            }
        }
        if (!kStripFft) {
            dif_inv_0<NF>(v, t, X);
            dif_warp_sync();
            dif_inv_1<NF>(v, t, X, tws);
        }
        gb.sync();
        if (!kStripFft) dif_inv_2<NF>(v, t, X, tws);
        // without the stores the condition is still evaluated at run time (ncols is never negative), so that what
        // feeds them cannot be optimised away
        if (live && (!kStripStore || a.ncols < 0)) {
            float2* col = a.out + ((size_t)b * 2 * a.ntile + kx) * NF + t;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                // y = e + conj(twist) o, as two fma chains
                const float2 tw_ = twist_e(e), o = c2get(v[e], 1);
                stg2(col + e * P, make_float2(fmaf(o.x, tw_.x, fmaf(o.y, tw_.y, v[e].re.x)), fmaf(o.y, tw_.x, fmaf(-o.x, tw_.y, v[e].im.x))));
            }
        }
    }
}
