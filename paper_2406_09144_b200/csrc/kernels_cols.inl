// kernels_cols.inl -- column passes (included inside namespace frs by kernels.cuh)

// ------------------------------------------------------------------------------------------------
struct ConvColsArgs {
    float2* t;            // [nb][ntile][NF][2] in place
    const float* wt;      // [nb][ntile][2][NF][2]
    int ntile, dbg;
    int items_per_batch;  // ceil(ntile / G)
    int nitems;           // items_per_batch * nb
    size_t t_bstride, w_bstride;
    const float4* tw;
    const float2* twist;  // exp(-2 pi i n/(2 NF))
};

// Group = 2 roles x P threads; role 0 owns the even output bins of the length-2NF transform of the
// zero-extended column, role 1 the odd bins (input pre-multiplied by twist^n).  After . W and the
// inverse transforms:  y[n] = IFFT_NF(E')[n] + conj(twist^n) IFFT_NF(O')[n].
template <int NF>
__global__ void __launch_bounds__(Geo<NF, 2>::THREADS, Geo<NF, 2>::MINB)
conv_cols_kernel(ConvColsArgs a) {
    using GEO = Geo<NF, 2>;
    constexpr int P = GEO::P;
    extern __shared__ float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / (2 * P), role = (threadIdx.x / P) & 1, p = threadIdx.x % P;
    float4* gb = smem4 + GEO::TW + (size_t)g * 2 * xbuf_len(NF);
    float4* buf = gb + role * xbuf_len(NF);
    float4* cb = gb + xbuf_len(NF);              // combine buffer = role 1's exchange buffer, [e][p]
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int m = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = m < a.ntile;
        float4* tile = reinterpret_cast<float4*>(a.t + b * a.t_bstride) + (size_t)m * NF;
        const float2* w = reinterpret_cast<const float2*>(a.wt + b * a.w_bstride) + ((size_t)m * 2 + role) * NF;

        float2 v[2][kE];
        if (live) {
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float4 x = ldg4(tile + p + e * P);
                v[0][e] = lo(x);
                v[1][e] = hi(x);
            }
            // L2 prefetch: this item's weights (needed after the forward transform), the next item's tile
            if ((p & 15) == 0) {
#pragma unroll
                for (int e = 0; e < kE; ++e) prefetch_l2(w + p + e * P);
            }
            const int nitem = item + gridDim.x;
            if (nitem < a.nitems && (p & 7) == 0 && role == 0) {
                const int nb_ = nitem / a.items_per_batch;
                const int nm = (nitem - nb_ * a.items_per_batch) * GEO::G + g;
                if (nm < a.ntile) {
                    const float4* nt = reinterpret_cast<const float4*>(a.t + nb_ * a.t_bstride) + (size_t)nm * NF;
#pragma unroll
                    for (int e = 0; e < kE; ++e) prefetch_l2(nt + p + e * P);
                }
            }
            if (role) {
#pragma unroll
                for (int e = 0; e < kE; ++e) {
                    const float2 tw = __ldg(a.twist + p + e * P);
                    v[0][e] = cmul(v[0][e], tw);
                    v[1][e] = cmul(v[1][e], tw);
                }
            }
        } else {
#pragma unroll
            for (int e = 0; e < kE; ++e) { v[0][e] = make_float2(0.f, 0.f); v[1][e] = make_float2(0.f, 0.f); }
        }
        if (!(a.dbg & 2)) pair_fft<NF, false>(v, p, buf, tws);
        if (live && !(a.dbg & 8)) {
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 ww = ldg2(reinterpret_cast<const float*>(w + p + e * P));
                v[0][e] = cscale(v[0][e], ww.x);
                v[1][e] = cscale(v[1][e], ww.y);
            }
        }
        if (!(a.dbg & 2)) pair_fft<NF, true>(v, p, buf, tws);
        if (role) {
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 tw = __ldg(a.twist + p + e * P);
                cb[e * P + p] = pack(cmulc(v[0][e], tw), cmulc(v[1][e], tw));
            }
        }
        __syncthreads();
        if (!role && live) {
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float4 o = cb[e * P + p];
                stg4(tile + p + e * P, make_float4(v[0][e].x + o.x, v[0][e].y + o.y, v[1][e].x + o.z, v[1][e].y + o.w));
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
struct HartColsArgs {
    const float2* t;      // [nb][ntile][NF][2], columns x = 0..nx/2 of the row-transformed field
    float* out;           // [nb][NF][nx]
    const float* mul;     // optional [nb][NF][nx]: out = mul * H + add
    const float* add;     // optional [nb][NF][nx]
    const float* offset;  // optional device [nb]: out = H + offset[b]   (mu)
    int nx;
    int items_per_batch, nitems;
    size_t t_bstride, img_bstride;
    const float4* tw;
};

// F[y][x] = column FFT; H[y][x] = Re F - Im F and H[(-y) mod ny][nx - x] = Re F + Im F  (reading R6)
template <int NF>
__global__ void __launch_bounds__(Geo<NF, 1>::THREADS, Geo<NF, 1>::MINB)
hart_cols_kernel(HartColsArgs a) {
    using GEO = Geo<NF, 1>;
    constexpr int P = GEO::P;
    extern __shared__ float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * xbuf_len(NF);
    const int ntile = a.nx / 4 + 1;
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int m = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = m < ntile;

        float2 v[2][kE];
        if (live) {
            const float4* tile = reinterpret_cast<const float4*>(a.t + b * a.t_bstride) + (size_t)m * NF;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float4 x = ldg4(tile + p + e * P);
                v[0][e] = lo(x);
                v[1][e] = hi(x);
            }
        } else {
#pragma unroll
            for (int e = 0; e < kE; ++e) { v[0][e] = make_float2(0.f, 0.f); v[1][e] = make_float2(0.f, 0.f); }
        }
        pair_fft<NF, false>(v, p, buf, tws);
        if (live) {
            const size_t base = b * a.img_bstride;
            const float off = a.offset ? __ldg(a.offset + b) : 0.f;
            const int half = a.nx / 2;
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const int y = p + e * P, ym = (NF - y) & (NF - 1);
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int x = 2 * m + c;
                    if (x > half) continue;
                    const float2 f = v[c][e];
                    size_t i0 = base + (size_t)y * a.nx + x;
                    float h0 = f.x - f.y + off;
                    if (a.mul) h0 *= __ldg(a.mul + i0);
                    if (a.add) h0 += __ldg(a.add + i0);
                    a.out[i0] = h0;
                    if (x > 0 && x < half) {
                        size_t i1 = base + (size_t)ym * a.nx + (a.nx - x);
                        float h1 = f.x + f.y + off;
                        if (a.mul) h1 *= __ldg(a.mul + i1);
                        if (a.add) h1 += __ldg(a.add + i1);
                        a.out[i1] = h1;
                    }
                }
            }
        }
        __syncthreads();
    }
}
