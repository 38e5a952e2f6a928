// kernels_cols.inl -- column passes (included inside namespace frs by kernels.cuh)

// ------------------------------------------------------------------------------------------------
struct ConvColsArgs {
    CUtensorMap tmap;     // column map of t (tmap.h)
    const float2* t;      // [nb][len/8+1][NF/2][8][2] block layout (tmap.h): input
    float2* out;          // [nb][2 ntile][NF]: output, column kx contiguous (whole-sector, coalesced stores)
    const float* wt;      // [nb][ntile][2 (column in tile)][NF (q)][2 (even, odd bin)]
    int ncols;            // columns that exist per batch (row length + 1)
    int ntile;            // tiles per batch
    int items_per_batch;  // ceil(ncols / G)
    int nitems;           // items_per_batch * nb
    size_t w_bstride;
    const float4* tw;
    const float2* twist;  // exp(-2 pi i n/(2 NF))
};

// One group (P threads) convolves ONE column: the pair of transforms a thread carries are the even
// and the odd output bins of the length-2NF transform of the zero-extended column,
//   even bins = FFT_NF(x),  odd bins = FFT_NF(x twist^n);   after . W and the inverse transforms
//   y[n] = IFFT_NF(E')[n] + conj(twist^n) IFFT_NF(O')[n]
// so input, twiddles and the final combination are all thread-local.
//
// Global reads never stall the arithmetic and cost no LSU instructions: one 8 NF-byte staging buffer
// per group is filled by the TMA unit (the weights by one bulk copy, the column -- 16-byte pieces at a
// 32-byte stride in the block layout -- by tensor copies that land it contiguously), alternately with
//   the weights of THIS item     (issued after the first exchange barrier of the forward transform --
//                                 every thread has picked up its samples by then -- and awaited
//                                 after the forward transform), and
//   the column of the NEXT item  (issued after the first exchange barrier of the inverse transform --
//                                 the weights have been consumed -- in flight during the rest of it).
template <int NF> struct ColsGeo : Geo<NF, 1, NF / 2> {};

template <int NF>
__global__ void __launch_bounds__(ColsGeo<NF>::THREADS, ColsGeo<NF>::MINB)
conv_cols_kernel(const __grid_constant__ ConvColsArgs a) {
    using GEO = ColsGeo<NF>;
    constexpr int P = GEO::P;
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    float2* stage = reinterpret_cast<float2*>(buf + xbuf_len(NF));                     // [NF] float2
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem4 + GEO::TW + (size_t)GEO::G * GEO::GROUP_SLOTS) + g;
    const GroupBar gb = GEO::bar(g);
    load_twiddles<NF>(tws, a.tw);
    if (p == 0) mbar_init(bar, 1);
    // twist^n for the thread's samples n = p + e P, from the exactly rounded table (a product of two
    // rounded factors costs a measurable part of the CG error budget and no time is gained by it)
    auto twist_e = [&](int e) { return __ldg(a.twist + p + e * P); };

    constexpr int BOXR = tma_box_pairs(NF), NCOPY = tma_col_copies(NF);
    auto column = [&](int item, bool& live, int& b, int& kx, const float*& w) {
        b = item / a.items_per_batch;
        kx = (item - b * a.items_per_batch) * GEO::G + g;
        live = item < a.nitems && kx < a.ncols;
        w = a.wt + b * a.w_bstride + (size_t)kx * NF * 2;
    };
    auto fetch_weights = [&](const void* src, bool live) {       // one bulk copy of 8 NF bytes into the staging buffer
        if (p == 0 && live) {
            fence_proxy_async();
            mbar_expect_tx(bar, NF * 8);
            bulk_g2s(stage, src, NF * 8, bar);
        }
        __syncwarp();   // the issuing lane must not be left behind a warp that spins on the mbarrier
    };
    auto fetch_column = [&](int b, int kx, bool live) {          // column kx lands as NF contiguous samples
        if (p == 0 && live) {
            fence_proxy_async();
            mbar_expect_tx(bar, NF * 8);
        }
        __syncwarp();
        if (p < NCOPY && live) tensor_g2s_5d(stage + 2 * BOXR * p, &a.tmap, 0, kx % kBlockBins, BOXR * p, kx / kBlockBins, b, bar);   // one copy per lane
        __syncwarp();
    };
    unsigned parity = 0;
    __syncthreads();
    {
        bool live; int b, kx; const float* w;
        column(blockIdx.x, live, b, kx, w);
        fetch_column(b, kx, live);
    }

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        bool live; int b, kx; const float* w;
        column(item, live, b, kx, w);

        C2 v[kE];
        if (live) {
            mbar_wait(bar, parity);
            parity ^= 1u;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 x = stage[p + e * P];
                v[e] = c2make(x, cmul(x, twist_e(e)));
            }
        } else {
#pragma unroll
            for (int e = 0; e < kE; ++e) v[e] = c2zero();
        }
        // forward transforms; the weights start to arrive behind the first barrier
        stage_compute<NF, 0, false>(v, p, tws);
        if constexpr (plan_stages(NF) > 1) stage_scatter2<NF, 0>(v, p, buf);
        gb.sync();
        fetch_weights(w, live);
        if constexpr (plan_stages(NF) > 1) {
            canon_gather2<NF>(v, p, buf);
            gb.sync();
            pair_fft_from<NF, false, 1>(v, p, buf, tws, gb);
        }
        if (live) {
            mbar_wait(bar, parity);
            parity ^= 1u;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 ww = stage[p + e * P];               // (even-bin weight, odd-bin weight)
                v[e].re = f2mul(v[e].re, ww);
                v[e].im = f2mul(v[e].im, ww);
            }
        }
        // inverse transforms; the next column starts to arrive behind the first barrier
        stage_compute<NF, 0, true>(v, p, tws);
        if constexpr (plan_stages(NF) > 1) stage_scatter2<NF, 0>(v, p, buf);
        gb.sync();
        {
            bool nlive; int nb_, nkx; const float* nw;
            column(item + gridDim.x, nlive, nb_, nkx, nw);
            fetch_column(nb_, nkx, nlive);
        }
        if constexpr (plan_stages(NF) > 1) {
            canon_gather2<NF>(v, p, buf);
            gb.sync();
            pair_fft_from<NF, true, 1>(v, p, buf, tws, gb);
        }
        if (live) {
            float2* col = a.out + ((size_t)b * 2 * a.ntile + kx) * NF + p;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                // y = e + conj(twist) o, as two fma chains
                const float2 t = twist_e(e), o = c2get(v[e], 1);
                stg2(col + e * P, make_float2(fmaf(o.x, t.x, fmaf(o.y, t.y, v[e].re.x)), fmaf(o.y, t.x, fmaf(-o.x, t.y, v[e].im.x))));
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
struct HartColsArgs {
    const float2* t;      // pair layout of tmap.h ([nb][m][NF/2][2][2]): columns x = 0..nx/2 of the row-transformed field (NF rows)
    float* out;           // [nb][nx][NF]  TRANSPOSED: out[x][y] = H[y][x]
    const float* mul;     // optional [nb][nx][NF]: out = mul * (H + offset) + add
    const float* add;     // optional [nb][nx][NF]
    const float* offset;  // optional device [nb]   (mu)
    double* dot_partials; // optional [gridDim.x]: sum over the CTA's outputs of out * add (fp64) -- <v, M v> of a CG step
    int nx;
    int exp_out;          // out = exp(...) (the sky of a single-field, single-channel model: A2 fused into A1's last pass)
    int items_per_batch, nitems;
    size_t img_bstride;
    const float4* tw;
};

// F[y][x] = column FFT; H[y][x] = Re F - Im F and H[(-y) mod NF][nx - x] = Re F + Im F  (reading R6).
// Column x of H is one contiguous run of the transposed output, so all stores are coalesced.
// Input: the column pair (2m, 2m+1) is one contiguous run of 16 NF bytes in the pair layout; lanes read neighbouring
// 8-byte samples (staging it through shared memory by a bulk or a tensor copy was measured 5-8 % slower: the landing
// costs a second trip through the shared-memory pipe and the copy can only start behind the transform).
// The epilogue variant is a template parameter: as run-time flags the 64-fold unrolled optional pieces (the predicated-off
// expf sequences alone) cost a third of the kernel's issue slots (measured: 113 us instead of 76 us per pass at 4096^2).
enum HartMode { kHPlain = 0,      // out = H + offset
                kHExp = 1,        // out = exp(H + offset)                        (sky of a single-field model)
                kHMul = 2,        // out = mul . H                                 (N'^-1: K^-1 in harmonic space; gradient without prior)
                kHMulAdd = 3,     // out = mul . H + add                           (gradient with prior)
                kHMulAddDot = 4 };// ... and sum out . add in fp64                 (last pass of a CG iteration)
template <int NF, int MODE>
__global__ void __launch_bounds__(RowsGeo<NF>::THREADS, RowsGeo<NF>::MINB)
hart_cols_kernel(const HartColsArgs a) {
    using GEO = RowsGeo<NF>;
    constexpr int P = GEO::P;
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    const int ntile = a.nx / 4 + 1;
    const GroupBar gb = GEO::bar(g);
    double dacc = 0.0;
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int m = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = m < ntile;

        C2 v[kE];
        if (live) {
            const float* c0 = reinterpret_cast<const float*>(a.t + b * spec_batch_stride(NF, a.nx / 2, kPairBins)
                                                             + spec_index(NF, 2 * m, 0, kPairBins));
            const bool two = 2 * m + 1 <= a.nx / 2;            // the last pair may hold one column only
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const int y = p + e * P;
                const float* q = c0 + 2 * ((y >> 1) * 4 + (y & 1));
                const float2 x0 = ldg2(q);
                const float2 x1 = two ? ldg2(q + 4) : make_float2(0.f, 0.f);
                v[e] = c2make(x0, x1);
            }
        } else {
#pragma unroll
            for (int e = 0; e < kE; ++e) v[e] = c2zero();
        }
        pair_fft<NF, false>(v, p, buf, tws, gb);
        if (live) {
            const size_t base = b * a.img_bstride;
            const float off = (MODE == kHPlain || MODE == kHExp) && a.offset ? __ldg(a.offset + b) : 0.f;
            const int half = a.nx / 2;
            constexpr bool MUL = MODE >= kHMul, ADD = MODE >= kHMulAdd;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int x = 2 * m + c;
                if (x > half) continue;
                const bool mirror = x > 0 && x < half;
                // column x of H: rows y (Re - Im); column nx - x: rows (-y) mod NF (Re + Im)
#pragma unroll
                for (int side = 0; side < 2; ++side) {
                    if (side == 1 && !mirror) continue;
                    const size_t col = base + (size_t)(side ? a.nx - x : x) * NF;
                    float mu[kE], ad[kE];
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        const int y = p + e * P, yy = side ? (NF - y) & (NF - 1) : y;
                        if (MUL) mu[e] = ldg1(a.mul + col + yy);
                        if (ADD) ad[e] = ldg1(a.add + col + yy);
                    }
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        const int y = p + e * P, yy = side ? (NF - y) & (NF - 1) : y;
                        const float2 f = c2get(v[e], c);
                        float h = (side ? f.x + f.y : f.x - f.y) + off;
                        if (MUL) h *= mu[e];
                        if (ADD) h += ad[e];
                        if (MODE == kHMulAddDot) dacc += (double)h * (double)ad[e];
                        if (MODE == kHExp) h = expf(h);
                        a.out[col + yy] = h;
                    }
                }
            }
        }
    }
    if (MODE == kHMulAddDot) {
        // fixed-order block reduction: warp shuffle tree, then warp 0 over the per-warp sums
        __shared__ double dred[32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dacc += __shfl_down_sync(0xffffffffu, dacc, o);
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) dred[w] = dacc;
        __syncthreads();
        if (w == 0) {
            const int nw = blockDim.x >> 5;
            double x = l < nw ? dred[l] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            if (l == 0) a.dot_partials[blockIdx.x] = x;
        }
    }
}
