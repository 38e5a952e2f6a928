// kernels_cols.inl -- column passes (included inside namespace frs by kernels.cuh)

// ------------------------------------------------------------------------------------------------
struct ConvColsArgs {
    float2* t;            // [nb][ntile][NF][2] in place
    const float* wt;      // [nb][ntile][2 (column in tile)][NF (q)][2 (even, odd bin)]
    int ntile;
    int items_per_batch;  // ceil(2 ntile / G)
    int nitems;           // items_per_batch * nb
    size_t t_bstride, w_bstride;
    const float4* tw;
    const float2* twist;  // exp(-2 pi i n/(2 NF))
};

// One group (P threads) convolves ONE column: the pair of transforms a thread carries are the even
// and the odd output bins of the length-2NF transform of the zero-extended column,
//   even bins = FFT_NF(x),  odd bins = FFT_NF(x twist^n);   after . W and the inverse transforms
//   y[n] = IFFT_NF(E')[n] + conj(twist^n) IFFT_NF(O')[n]
// so input, twiddles and the final combination are all thread-local.  Work item = (tile, column);
// the two columns of a tile go to neighbouring CTAs, which share the tile's sectors through L2.
//
// Global reads never stall the arithmetic: one 8 NF-byte staging buffer per group is time-shared by
//   the column of the NEXT item  (cp.async, every thread copies exactly the 16 samples it will use, so
//                                 no barrier is needed; issued once the weights have been consumed,
//                                 in flight during the inverse transforms), and
//   the weights of THIS item     (one bulk TMA copy of the contiguous 8 NF-byte weight column, issued
//                                 after the first exchange barrier of the forward transform -- every
//                                 thread has picked up its samples by then -- and awaited on an
//                                 mbarrier after the forward transform).
template <int NF> struct ColsGeo : Geo<NF, 1, NF / 2> {};

template <int NF>
__global__ void __launch_bounds__(ColsGeo<NF>::THREADS, ColsGeo<NF>::MINB)
conv_cols_kernel(ConvColsArgs a) {
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

    auto column = [&](int item, bool& live, float2*& col, const float*& w) {
        const int b = item / a.items_per_batch;
        const int mc = (item - b * a.items_per_batch) * GEO::G + g;      // 2 m + c
        live = item < a.nitems && mc < 2 * a.ntile;
        col = a.t + b * a.t_bstride + (size_t)(mc >> 1) * NF * 2 + (mc & 1);      // stride 2 float2 per row
        w = a.wt + b * a.w_bstride + (size_t)mc * NF * 2;
    };
    auto stage_column = [&](int item) {
        bool live; float2* col; const float* w;
        column(item, live, col, w);
        if (live) {
#pragma unroll
            for (int e = 0; e < kE; ++e) cp_async8(stage + p + e * P, col + 2 * (p + e * P));
        }
        cp_async_commit();
    };
    stage_column(blockIdx.x);
    __syncthreads();
    unsigned parity = 0;

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        bool live; float2* col; const float* w;
        column(item, live, col, w);

        C2 v[kE];
        cp_async_wait_all();
        if (live) {
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
        if constexpr (plan_stages(NF) > 1) {
            stage_scatter2<NF, 0>(v, p, buf);
            gb.sync();
        } else {
            gb.sync();
        }
        if (p == 0 && live) {
            fence_proxy_async();
            mbar_expect_tx(bar, NF * 8);
            bulk_g2s(stage, w, NF * 8, bar);
        }
        __syncwarp();   // the issuing lane must not be left behind a warp that spins on the mbarrier
        if constexpr (plan_stages(NF) > 1) {
            canon_gather2<NF>(v, p, buf);
            gb.sync();
            pair_fft_from<NF, false, 1>(v, p, buf, tws, gb);
        }
        if (live) {
            mbar_wait(bar, parity);
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 ww = stage[p + e * P];               // (even-bin weight, odd-bin weight)
                v[e].re = f2mul(v[e].re, ww);
                v[e].im = f2mul(v[e].im, ww);
            }
            parity ^= 1u;
        }
        // the staging slots a thread has just read are its own: refill them with the next column
        stage_column(item + gridDim.x);
        pair_fft<NF, true>(v, p, buf, tws, gb);
        if (live) {
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 o = cmulc(c2get(v[e], 1), twist_e(e));
                stg2(col + 2 * (p + e * P), make_float2(v[e].re.x + o.x, v[e].im.x + o.y));
            }
        }
    }
    cp_async_wait_all();
}

// ------------------------------------------------------------------------------------------------
struct HartColsArgs {
    const float2* t;      // [nb][ntile][NF][2], columns x = 0..nx/2 of the row-transformed field (NF rows)
    float* out;           // [nb][nx][NF]  TRANSPOSED: out[x][y] = H[y][x]
    const float* mul;     // optional [nb][nx][NF]: out = mul * (H + offset) + add
    const float* add;     // optional [nb][nx][NF]
    const float* offset;  // optional device [nb]   (mu)
    int nx;
    int items_per_batch, nitems;
    size_t t_bstride, img_bstride;
    const float4* tw;
};

// F[y][x] = column FFT; H[y][x] = Re F - Im F and H[(-y) mod NF][nx - x] = Re F + Im F  (reading R6).
// Column x of H is one contiguous run of the transposed output, so all stores are coalesced.
template <int NF>
__global__ void __launch_bounds__(RowsGeo<NF>::THREADS, RowsGeo<NF>::MINB)
hart_cols_kernel(HartColsArgs a) {
    using GEO = RowsGeo<NF>;
    constexpr int P = GEO::P;
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    const int ntile = a.nx / 4 + 1;
    const GroupBar gb = GEO::bar(g);
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int m = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = m < ntile;

        C2 v[kE];
        if (live) {
            const float4* tile = reinterpret_cast<const float4*>(a.t + b * a.t_bstride) + (size_t)m * NF;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float4 x = ldg4(tile + p + e * P);
                v[e] = c2make(make_float2(x.x, x.y), make_float2(x.z, x.w));
            }
        } else {
#pragma unroll
            for (int e = 0; e < kE; ++e) v[e] = c2zero();
        }
        pair_fft<NF, false>(v, p, buf, tws, gb);
        if (live) {
            const size_t base = b * a.img_bstride;
            const float off = a.offset ? __ldg(a.offset + b) : 0.f;
            const int half = a.nx / 2;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int x = 2 * m + c;
                if (x > half) continue;
                const bool mirror = x > 0 && x < half;
                const size_t col0 = base + (size_t)x * NF, col1 = base + (size_t)(a.nx - x) * NF;
#pragma unroll
                for (int e = 0; e < kE; ++e) {
                    const int y = p + e * P, ym = (NF - y) & (NF - 1);
                    const float2 f = c2get(v[e], c);
                    float h0 = f.x - f.y + off;
                    if (a.mul) h0 *= ldg1(a.mul + col0 + y);
                    if (a.add) h0 += ldg1(a.add + col0 + y);
                    a.out[col0 + y] = h0;
                    if (mirror) {
                        float h1 = f.x + f.y + off;
                        if (a.mul) h1 *= ldg1(a.mul + col1 + ym);
                        if (a.add) h1 += ldg1(a.add + col1 + ym);
                        a.out[col1 + ym] = h1;
                    }
                }
            }
        }
        gb.sync();
    }
}
