// kernels_inv.inl -- inverse row pass of the convolution (included inside namespace frs by kernels.cuh)

enum RowsInvMode { kPlain = 0, kMulS = 1, kEnergy = 2 };

struct RowsInvArgs {
    const float2* t;      // [nb][ntile][ny][2]
    float* out;           // [nb][ny][NF]
    const float* s;       // [nb][ny][NF]  (kMulS, kEnergy)
    const float* j;       // [nb][ny][NF]  (kEnergy)
    double* partials;     // [gridDim.x][2]  (kEnergy): sum s*c, sum j*s
    int ny, mode, dbg;
    int items_per_batch, nitems;
    size_t t_bstride, img_bstride;
    const float4* tw;
    const float2* twist;
};

template <int NF>
__global__ void __launch_bounds__(Geo<NF, 1>::THREADS, Geo<NF, 1>::MINB)
rows_inv_kernel(RowsInvArgs a) {
    using GEO = Geo<NF, 1>;
    constexpr int P = GEO::P;
    constexpr int NTILE = NF / 2 + 1;
    extern __shared__ float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * xbuf_len(NF);
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();
    double acc_sc = 0.0, acc_js = 0.0;

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = 2 * rp < a.ny;
        const int y0 = 2 * rp;

        if (live) {
            const float4* tb = reinterpret_cast<const float4*>(a.t + b * a.t_bstride);
            float4 r0[kE / 2], r1[kE / 2];
#pragma unroll
            for (int i = 0; i < kE / 2; ++i) {
                const float4* q = (a.dbg & 1) ? tb + ((size_t)rp * (NF / 2) + p + i * P) * 2 : tb + (size_t)(p + i * P) * a.ny + y0;
                r0[i] = ldg4(q);
                r1[i] = ldg4(q + 1);
            }
#pragma unroll
            for (int i = 0; i < kE / 2; ++i) {
                const int k = 2 * (p + i * P);
                buf[xpad(k)] = make_float4(r0[i].x, r0[i].y, r1[i].x, r1[i].y);
                buf[xpad(k + 1)] = make_float4(r0[i].z, r0[i].w, r1[i].z, r1[i].w);
            }
            if (p == 0) {                               // tail tile: column NF
                const float4* q = tb + (size_t)(NTILE - 1) * a.ny + y0;
                const float4 t0 = ldg4(q), t1 = ldg4(q + 1);
                buf[xpad(NF)] = make_float4(t0.x, t0.y, t1.x, t1.y);
            }
        }
        __syncthreads();
        // Z'[k] = (Y[k] + conj Y[NF-k]) + i conj(twist[k]) (Y[k] - conj Y[NF-k]),  k = 0..NF-1
        float2 v[2][kE];
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int k = p + e * P;
            const float2 w = __ldg(a.twist + k);
            float4 yk = make_float4(0.f, 0.f, 0.f, 0.f), yn = yk;
            if (live) { yk = buf[xpad(k)]; yn = buf[xpad(NF - k)]; }
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const float2 ya = t ? hi(yk) : lo(yk), ym = cconj(t ? hi(yn) : lo(yn));
                const float2 s = cadd(ya, ym), d = cmulc(csub(ya, ym), w);
                v[t][e] = make_float2(s.x - d.y, s.y + d.x);
            }
        }
        __syncthreads();
        if (!(a.dbg & 2)) pair_fft<NF, true>(v, p, buf, tws);

        if (live) {
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const size_t row = b * a.img_bstride + (size_t)(y0 + t) * NF;
#pragma unroll
                for (int e = 0; e < kE / 2; ++e) {
                    const int n = p + e * P;
                    float2 c = v[t][e];
                    if (a.dbg & 4) {
                    } else if (a.mode == kMulS) {
                        const float2 s = ldg2(a.s + row + 2 * n);
                        c.x *= s.x; c.y *= s.y;
                    } else if (a.mode == kEnergy) {
                        const float2 s = ldg2(a.s + row + 2 * n), j = ldg2(a.j + row + 2 * n);
                        acc_sc += (double)s.x * (double)c.x + (double)s.y * (double)c.y;
                        acc_js += (double)j.x * (double)s.x + (double)j.y * (double)s.y;
                        c.x = s.x * (c.x - j.x); c.y = s.y * (c.y - j.y);
                    }
                    stg2(a.out + row + 2 * n, c);
                }
            }
        }
        __syncthreads();
    }
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
