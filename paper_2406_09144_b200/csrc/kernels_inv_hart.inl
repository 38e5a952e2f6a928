// kernels_inv_hart.inl -- inverse row pass of the convolution FUSED with the row pass of the Hartley transform that
// follows it in the latent-space path (included inside namespace frs by kernels.cuh).
//
// In the gradient and in the metric apply the convolution's last pass writes  acc = s . C(...)  [rows][NF] and the adjoint
// correlated-field transform starts with a real-to-complex row pass over the very same rows.  The NF/2 complex samples a
// row keeps after the crop, z[n] = y[2n] + i y[2n+1], n < NF/2, ARE the packed input of that row pass, and they are
// still in registers: thread p holds n = p + P e, e < 8.  So the rows are not written and read back (2 x 4 NF^2 bytes
// and one kernel of the latency-bound kind): they are redistributed once through shared memory to the P/2 threads that
// carry the half-length transform (16 elements each), transformed, unpacked (kernels.cuh, rows_fwd) and stored in the
// pair layout hart_cols reads.  The inverse pass waits for its TMA gather a third of the time (profiles/): the half-
// length transform runs in that shadow -- the other half of the threads has already moved on to the next row pair.
struct RowsInvHartArgs {
    RowsInvArgs inv;        // the inverse pass (out unused)
    float2* th;             // [nb][NF/4+1][rows/2][2][2]: pair layout of tmap.h
    float scale;            // 0.5 x sign of the Hartley row pass
    const float4* tw2;      // stage twiddles of length NF/2
    const float2* twist2;   // exp(-2 pi i k / NF), k = 0..NF/2
};

template <int NF> struct RowsInvHartGeo : Geo<NF, 1, 0, 256> {
    using B = Geo<NF, 1, 0, 256>;
    static constexpr int NF2 = NF / 2, P2 = B::P / 2;
    static constexpr int TW2 = (plan_tw_total(NF2) + 7) & ~7;
    static constexpr int FBUF = xbuf_len(NF2);
    static constexpr int GROUP_SLOTS = B::GROUP_SLOTS + FBUF;
    static constexpr int SMEM = (B::TW + TW2 + B::G * GROUP_SLOTS + B::BAR_SLOTS) * (int)sizeof(float4);
    static_assert(P2 % 32 == 0, "the half-length transform needs whole warps");
};

template <int NF, int MODE>
__global__ void __launch_bounds__(RowsInvHartGeo<NF>::THREADS, RowsInvHartGeo<NF>::MINB)
rows_inv_hart_kernel(const __grid_constant__ RowsInvHartArgs aa) {
    using GEO = RowsInvHartGeo<NF>;
    static_assert(MODE == kMulS || MODE == kEnergy, "fused variants: . s and the energy epilogue");
    const RowsInvArgs& a = aa.inv;
    constexpr int P = GEO::P, NF2 = GEO::NF2, P2 = GEO::P2;
    constexpr int BOX = tma_box_bins(NF), NOPS = tma_bin_copies(NF);
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    float4* tws2 = smem4 + GEO::TW;
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + GEO::TW2 + (size_t)g * GEO::GROUP_SLOTS;
    float4* fbuf = buf + xbuf_len(NF);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem4 + GEO::TW + GEO::TW2 + (size_t)GEO::G * GEO::GROUP_SLOTS) + g;
    const GroupBar gb = GEO::bar(g);
    const GroupBar fb = GroupBar{1 + GEO::G + g, P2};          // the threads of the half-length transform
    load_twiddles<NF>(tws, a.tw);
    load_twiddles<NF2>(tws2, aa.tw2);
    if (p == 0) mbar_init(bar, 1);
    __syncthreads();
    double acc_sc = 0.0, acc_js = 0.0;
    unsigned parity = 0;

    auto gather = [&](int item) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = item < a.nitems && 2 * rp < a.ny;
        if (live && p == 0) {
            fence_proxy_async();
            mbar_expect_tx(bar, NOPS * BOX * 16);
        }
        __syncwarp();
        if (live && p < 32)
            for (int j = p; j < NOPS; j += 32) tensor_g2s_3d(buf + BOX * j, &a.tmap, 4 * rp, BOX * j, b, bar);
        __syncwarp();
        if (live) {
            const size_t row = b * a.img_bstride + (size_t)(2 * rp) * NF;
            prefetch_l2(a.s + row + 32 * p);
            if (MODE == kEnergy) prefetch_l2(a.j + row + 32 * p);
        }
    };
    gather(blockIdx.x);

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int b = item / a.items_per_batch;
        const int rp = (item - b * a.items_per_batch) * GEO::G + g;
        const bool live = 2 * rp < a.ny;
        const int y0 = 2 * rp;

        if (live) { mbar_wait(bar, parity); parity ^= 1u; }
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

        // epilogue on the kept half (samples 2n, 2n+1 of row t are the components of z_t[n], n = p + e P, e < 8)
        if (live) {
            const size_t row0 = b * a.img_bstride + (size_t)y0 * NF;
            float2 sv[2][kE / 2], jv[2][kE / 2];
#pragma unroll
            for (int t = 0; t < 2; ++t)
#pragma unroll
                for (int e = 0; e < kE / 2; ++e) sv[t][e] = ldg2(a.s + row0 + (size_t)t * NF + 2 * (p + e * P));
            if (MODE == kEnergy) {
#pragma unroll
                for (int t = 0; t < 2; ++t)
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) jv[t][e] = ldg2(a.j + row0 + (size_t)t * NF + 2 * (p + e * P));
            }
#pragma unroll
            for (int e = 0; e < kE / 2; ++e) {
                float2 c[2];
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    c[t] = c2get(v[e], t);
                    if (MODE == kMulS) {
                        c[t].x *= sv[t][e].x; c[t].y *= sv[t][e].y;
                    } else {
                        const float2 s = sv[t][e], j = jv[t][e];
                        acc_sc += (double)s.x * (double)c[t].x + (double)s.y * (double)c[t].y;
                        acc_js += (double)j.x * (double)s.x + (double)j.y * (double)s.y;
                        c[t].x = s.x * (c[t].x - j.x); c[t].y = s.y * (c[t].y - j.y);
                    }
                }
                v[e] = c2make(c[0], c[1]);
            }
        }
        // hand the NF/2 packed samples to the P/2 threads of the half-length transform: dense slot n = p + e P.
        // (fbuf is free: its previous users have passed the group barriers of this item)
#pragma unroll
        for (int e = 0; e < kE / 2; ++e) fbuf[p + e * P] = pack(live ? v[e] : c2zero());
        gb.sync();
        if (p >= P2) continue;                    // on to the next row pair (they wait at its first group barrier)

        C2 u[kE];
#pragma unroll
        for (int e = 0; e < kE; ++e) u[e] = unpack(fbuf[p + e * P2]);
        fb.sync();                                // everyone has its samples: the exchanges may overwrite fbuf
        pair_fft<NF2, false>(u, p, fbuf, tws2, fb);
#pragma unroll
        for (int e = 0; e < kE; ++e) fbuf[p + e * P2] = pack(u[e]);      // park Z densely for the mirror reads
        fb.sync();
        C2 xn = c2zero();
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int k = p + e * P2;
            const C2 zm = unpack(fbuf[(NF2 - k) & (NF2 - 1)]);
            const float2 w0 = __ldg(aa.twist2 + k);
            const float2 w = make_float2(w0.x * aa.scale, w0.y * aa.scale);
            const float2 sc = f2bc(aa.scale);
            C2 s, d0;
            s.re = f2add(u[e].re, zm.re);  s.im = f2sub(u[e].im, zm.im);
            d0.re = f2sub(u[e].re, zm.re); d0.im = f2add(u[e].im, zm.im);
            const C2 d = c2mul_dir<false>(d0, w);
            if (e == 0 && p == 0) {
                xn.re = f2fma(s.re, sc, f2neg(d.im));
                xn.im = f2fma(s.im, sc, d.re);
            }
            u[e].re = f2fma(s.re, sc, d.im);
            u[e].im = f2fma(s.im, sc, f2neg(d.re));
        }
        fb.sync();                                // every mirror slot has been read
        if (live) {
            auto slot = [](const C2& x) { return make_float4(x.re.x, x.im.x, x.re.y, x.im.y); };
            float4* ob = reinterpret_cast<float4*>(aa.th + b * spec_batch_stride(a.ny, NF2, kPairBins));
#pragma unroll
            for (int e = 0; e < kE; ++e) stg4(ob + spec_index(a.ny, p + e * P2, y0, kPairBins) / 2, slot(u[e]));
            if (p == 0) stg4(ob + spec_index(a.ny, NF2, y0, kPairBins) / 2, slot(xn));
        }
    }
    if (MODE == kEnergy) {
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
