#include "launch.h"
namespace frs {
template <int NF>
static int run(cudaStream_t st, const ConvColsArgs& a0, int nb) {
    using GEO = ColsGeo<NF>;
    static int ctas = 0;
    if (!ctas) {
        cudaError_t e = set_smem(conv_cols_kernel<NF>, GEO::SMEM);
        if (e != cudaSuccess) return (int)e;
        ctas = resident_ctas(conv_cols_kernel<NF>, GEO::THREADS, GEO::SMEM);
        if (!ctas) return (int)cudaErrorUnknown;
    }
    ConvColsArgs a = a0;
    a.items_per_batch = (a.ncols + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
    conv_cols_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_conv_cols(cudaStream_t st, int nf, const ConvColsArgs& a, int nb) {
#define CALL(N) return run<N>(st, a, nb)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
