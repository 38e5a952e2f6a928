#include "launch.h"
namespace frs {
template <int NF>
static int run(cudaStream_t st, const ConvColsArgs& a, int nb) {
    using GEO = Geo<NF, 2>;
    static bool attr = false;
    if (!attr) { cudaError_t e = set_smem(conv_cols_kernel<NF>, GEO::SMEM); if (e != cudaSuccess) return (int)e; attr = true; }
    dim3 grid((a.ntile + GEO::G - 1) / GEO::G, nb);
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
