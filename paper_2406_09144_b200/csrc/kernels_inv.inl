// kernels_inv.inl -- inverse row pass of the convolution (included inside namespace frs by kernels.cuh)

enum RowsInvMode { kPlain = 0, kMulS = 1, kEnergy = 2 };

struct RowsInvArgs {
    const float2* t;      // [nb][ntile][ny][2]
    float* out;           // [nb][ny][NF]
    const float* s;       // [nb][ny][NF]  (kMulS, kEnergy)
    const float* j;       // [nb][ny][NF]  (kEnergy)
    double* partials;     // [gridDim.x][2]  (kEnergy): sum s*c, sum j*s
    int ny, mode;
    int items_per_batch, nitems;
    size_t t_bstride, img_bstride;
    const float4* tw;
    const float2* twist;
};

// Pipeline: the half-spectrum rows of the NEXT item are gathered by 16-byte cp.async copies straight
// into the exchange buffer as soon as the transform has left it (before its last, register-only
// stage), so the gather is in flight during that stage and the epilogue.  Landing layout:
// slot r*(NF/2+1) + m = (Y_r[2m], Y_r[2m+1]) for row r of the pair.
template <int NF>
__global__ void __launch_bounds__(RowsGeo<NF>::THREADS, RowsGeo<NF>::MINB)
rows_inv_kernel(RowsInvArgs a) {
    using GEO = RowsGeo<NF>;
    constexpr int P = GEO::P;
    constexpr int NTILE = NF / 2 + 1;
    extern __shared__ float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    const float2* land = reinterpret_cast<const float2*>(buf);      // Y_r[k] at land[r*2*NTILE + k]
    const GroupBar gb = GEO::bar(g);
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();
    double acc_sc = 0.0, acc_js = 0.0;

    auto gather = [&](int item) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        if (item < a.nitems && 2 * rp < a.ny) {
            const float4* tb = reinterpret_cast<const float4*>(a.t + b * a.t_bstride) + 2 * rp;
            // lanes (2j, 2j+1) fetch rows (0, 1) of the same tile: one 32-byte sector per lane pair
            const int r = p & 1;
#pragma unroll
            for (int i = 0; i < kE; ++i) {
                const int m = (p >> 1) + i * (P / 2);
                cp_async16(buf + r * NTILE + m, tb + (size_t)m * a.ny + r);
            }
            if (p < 2) cp_async16(buf + r * NTILE + NTILE - 1, tb + (size_t)(NTILE - 1) * a.ny + r);
            // warm L2 with the rows of s (and j) the epilogue of that item will read: P lines of 128 B
            if (a.mode != kPlain) {
                const size_t row = b * a.img_bstride + (size_t)(2 * rp) * NF;
                prefetch_l2(a.s + row + 32 * p);
                if (a.mode == kEnergy) prefetch_l2(a.j + row + 32 * p);
            }
        }
        cp_async_commit();
    };
    gather(blockIdx.x);

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = 2 * rp < a.ny;
        const int y0 = 2 * rp;

        cp_async_wait_all();
        gb.sync();
        // Z'[k] = (Y[k] + conj Y[NF-k]) + i conj(twist[k]) (Y[k] - conj Y[NF-k]),  k = 0..NF-1
        C2 v[kE];
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int k = p + e * P;
            const float2 w = __ldg(a.twist + k);
            float2 z[2];
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                float2 ya = make_float2(0.f, 0.f), ym = ya;
                if (live) { ya = land[t * 2 * NTILE + k]; ym = cconj(land[t * 2 * NTILE + NF - k]); }
                const float2 s = cadd(ya, ym), d = cmulc(csub(ya, ym), w);
                z[t] = make_float2(s.x - d.y, s.y + d.x);
            }
            v[e] = c2make(z[0], z[1]);
        }
        gb.sync();
        pair_fft_head<NF, true>(v, p, buf, tws, gb);
        gather(item + gridDim.x);                 // buf is free from here to the top of the loop
        pair_fft_tail<NF, true>(v, p, tws);

        if (live) {
            const size_t row0 = b * a.img_bstride + (size_t)y0 * NF;
            float2 sv[2][kE / 2], jv[2][kE / 2];
            if (a.mode != kPlain) {
#pragma unroll
                for (int t = 0; t < 2; ++t)
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) sv[t][e] = ldg2(a.s + row0 + (size_t)t * NF + 2 * (p + e * P));
            }
            if (a.mode == kEnergy) {
#pragma unroll
                for (int t = 0; t < 2; ++t)
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) jv[t][e] = ldg2(a.j + row0 + (size_t)t * NF + 2 * (p + e * P));
            }
#pragma unroll
            for (int t = 0; t < 2; ++t) {
#pragma unroll
                for (int e = 0; e < kE / 2; ++e) {
                    float2 c = c2get(v[e], t);
                    if (a.mode == kMulS) {
                        c.x *= sv[t][e].x; c.y *= sv[t][e].y;
                    } else if (a.mode == kEnergy) {
                        const float2 s = sv[t][e], j = jv[t][e];
                        acc_sc += (double)s.x * (double)c.x + (double)s.y * (double)c.y;
                        acc_js += (double)j.x * (double)s.x + (double)j.y * (double)s.y;
                        c.x = s.x * (c.x - j.x); c.y = s.y * (c.y - j.y);
                    }
                    stg2(a.out + row0 + (size_t)t * NF + 2 * (p + e * P), c);
                }
            }
        }
    }
    cp_async_wait_all();
    if (a.mode == kEnergy) {
        // fixed-order block reduction: warp shuffle tree, then warp 0 over the per-warp sums
        __shared__ double red[2][32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc_sc += __shfl_down_sync(0xffffffffu, acc_sc, o);
            acc_js += __shfl_down_sync(0xffffffffu, acc_js, o);
        }
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) { red[0][w] = acc_sc; red[1][w] = acc_js; }
        __syncthreads();
        if (w == 0) {
            const int nw = blockDim.x >> 5;
            double x = l < nw ? red[0][l] : 0.0, y = l < nw ? red[1][l] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                x += __shfl_down_sync(0xffffffffu, x, o);
                y += __shfl_down_sync(0xffffffffu, y, o);
            }
            if (l == 0) { a.partials[2 * blockIdx.x] = x; a.partials[2 * blockIdx.x + 1] = y; }
        }
    }
}
