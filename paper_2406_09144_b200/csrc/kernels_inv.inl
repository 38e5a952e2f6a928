// kernels_inv.inl -- inverse row pass of the convolution (included inside namespace frs by kernels.cuh)

enum RowsInvMode { kPlain = 0, kMulS = 1, kEnergy = 2, kResid = 3 };   // kResid: out = j - c (residual of Eq. 9)

struct RowsInvArgs {
    CUtensorMap tmap;     // columns map of t (tmap.h)
    const float2* t;      // [nb][cols][ny]: column kx contiguous (written by conv_cols)
    int cols;             // allocated columns per batch
    float* out;           // [nb][ny][NF]
    const float* s;       // [nb][ny][NF]  (kMulS, kEnergy)
    const float* j;       // [nb][ny][NF]  (kEnergy, kResid)
    double* partials;     // [gridDim.x][2]  (kEnergy): sum s*c, sum j*s
    int ny, mode;
    int items_per_batch, nitems;
    size_t img_bstride;
    const float4* tw;
    const float2* twist;
};

// Pipeline: the half spectrum of the NEXT row pair is gathered by the TMA unit (17 tensor copies of
// 16-byte pieces of the column-contiguous array conv_cols wrote, tmap.h: no LSU instructions) straight into the
// exchange buffer as soon as the transform has left it (before its last, register-only stage), so
// the gather is in flight during that stage and the epilogue.  Landing layout: dense 16-byte slots,
// slot k = (Y_0[k], Y_1[k]) of the two rows, k = 0..NF.
// MODE is a template parameter: the energy epilogue needs 32 more registers than the others and would
// make every variant spill.
template <int NF, int MODE>
__global__ void __launch_bounds__(RowsGeo<NF>::THREADS, RowsGeo<NF>::MINB)
rows_inv_kernel(const __grid_constant__ RowsInvArgs a) {
    using GEO = RowsGeo<NF>;
    constexpr int P = GEO::P;
    constexpr bool USE_TMA = tma_rows_ok(NF);      // smaller rows: boxes below the 128-byte TMA alignment -> cp.async
    constexpr int BOX = tma_box_bins(NF), NOPS = tma_bin_copies(NF);
    static_assert(BOX * NOPS <= xbuf_len(NF), "landing area exceeds the exchange buffer");
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + (size_t)g * GEO::GROUP_SLOTS;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem4 + GEO::TW + (size_t)GEO::G * GEO::GROUP_SLOTS) + g;
    const GroupBar gb = GEO::bar(g);
    load_twiddles<NF>(tws, a.tw);
    if (p == 0) mbar_init(bar, 1);
    __syncthreads();
    double acc_sc = 0.0, acc_js = 0.0;
    unsigned parity = 0;

    auto gather = [&](int item) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = item < a.nitems && 2 * rp < a.ny;
        if (live && !USE_TMA) {
            const float4* tb = reinterpret_cast<const float4*>(a.t + ((size_t)b * a.cols) * a.ny) + rp;
            for (int k = p; k <= NF; k += P) cp_async16(buf + k, tb + (size_t)k * (a.ny / 2));
        }
        if (!USE_TMA) cp_async_commit();
        if (live && USE_TMA && p == 0) {
            fence_proxy_async();
            mbar_expect_tx(bar, NOPS * BOX * 16);
        }
        if (P >= 32) __syncwarp();
        if (live && USE_TMA && p < 32)                                // the copies are spread over the first lanes
            for (int j = p; j < NOPS; j += (P < 32 ? P : 32)) tensor_g2s_3d(buf + BOX * j, &a.tmap, 4 * rp, BOX * j, b, bar);
        if (P >= 32) __syncwarp();
        if (live) {
            // warm L2 with the rows of s (and j) the epilogue of that item will read: P lines of 128 B
            if (MODE != kPlain) {
                const size_t row = b * a.img_bstride + (size_t)(2 * rp) * NF;
                if (MODE != kResid) prefetch_l2(a.s + row + 32 * p);
                if (MODE == kEnergy || MODE == kResid) prefetch_l2(a.j + row + 32 * p);
            }
        }
    };
    gather(blockIdx.x);

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = 2 * rp < a.ny;
        const int y0 = 2 * rp;

        if (USE_TMA) {
            if (live) { mbar_wait(bar, parity); parity ^= 1u; }
        } else {
            cp_async_wait_all();
            gb.sync();
        }
        // Z'[k] = (Y[k] + conj Y[NF-k]) + i conj(twist[k]) (Y[k] - conj Y[NF-k]),  k = 0..NF-1
        C2 v[kE];
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int k = p + e * P;
            const float2 w = __ldg(a.twist + k);
            if (live) {
                const float4 qa = buf[k], qm = buf[NF - k];
                const C2 ya = c2make(make_float2(qa.x, qa.y), make_float2(qa.z, qa.w));
                const C2 ym = c2make(make_float2(qm.x, qm.y), make_float2(qm.z, qm.w));
                C2 s, d0;
                s.re = f2add(ya.re, ym.re);  s.im = f2sub(ya.im, ym.im);
                d0.re = f2sub(ya.re, ym.re); d0.im = f2add(ya.im, ym.im);
                const C2 d = c2mul_dir<true>(d0, w);
                v[e].re = f2sub(s.re, d.im);
                v[e].im = f2add(s.im, d.re);
            } else {
                v[e] = c2zero();
            }
        }
        gb.sync();
        pair_fft_head<NF, true>(v, p, buf, tws, gb);
        gather(item + gridDim.x);                 // buf is free from here to the top of the loop
        pair_fft_tail<NF, true>(v, p, tws);

        if (live) {
            const size_t row0 = b * a.img_bstride + (size_t)y0 * NF;
            float2 sv[2][kE / 2], jv[2][kE / 2];
            if (MODE == kMulS || MODE == kEnergy) {
#pragma unroll
                for (int t = 0; t < 2; ++t)
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) sv[t][e] = ldg2(a.s + row0 + (size_t)t * NF + 2 * (p + e * P));
            }
            if (MODE == kEnergy || MODE == kResid) {
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
                    if (MODE == kMulS) {
                        c.x *= sv[t][e].x; c.y *= sv[t][e].y;
                    } else if (MODE == kEnergy) {
                        const float2 s = sv[t][e], j = jv[t][e];
                        acc_sc += (double)s.x * (double)c.x + (double)s.y * (double)c.y;
                        acc_js += (double)j.x * (double)s.x + (double)j.y * (double)s.y;
                        c.x = s.x * (c.x - j.x); c.y = s.y * (c.y - j.y);
                    } else if (MODE == kResid) {
                        c.x = jv[t][e].x - c.x; c.y = jv[t][e].y - c.y;
                    }
                    stg2(a.out + row0 + (size_t)t * NF + 2 * (p + e * P), c);
                }
            }
        }
    }
    cp_async_wait_all();
    if (MODE == kEnergy) {
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
