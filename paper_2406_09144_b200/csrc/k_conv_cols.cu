#include "launch.h"
namespace frs {
template <int NF>
static int run(cudaStream_t st, const ConvColsArgs& a0, int nb) {
    using GEO = ColsGeo<NF>;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, conv_cols_kernel<NF>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    ConvColsArgs a = a0;
    a.items_per_batch = (a.ncols + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
    conv_cols_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
template <int NF>
static int run_dif(cudaStream_t st, const ConvColsArgs& a0, int nb) {
    using GEO = ColsDifGeo<NF>;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, conv_cols_dif_kernel<NF>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    ConvColsArgs a = a0;
    a.items_per_batch = (a.ncols + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
    conv_cols_dif_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_conv_cols(cudaStream_t st, int nf, const ConvColsArgs& a, int nb) {
    switch (nf) {
        case 16: return run<16>(st, a, nb);
        case 32: return run<32>(st, a, nb);
        case 64: return run<64>(st, a, nb);
        case 128: return run<128>(st, a, nb);
        case 256: return run_dif<256>(st, a, nb);
        case 512: return run_dif<512>(st, a, nb);
        case 1024: return run_dif<1024>(st, a, nb);
        case 2048: return run_dif<2048>(st, a, nb);
        case 4096: return run_dif<4096>(st, a, nb);
        default: return (int)cudaErrorInvalidValue;
    }
}
}  // namespace frs
