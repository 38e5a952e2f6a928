#include "launch.h"
namespace frs {
template <int NF>
static int run(cudaStream_t st, const HartColsArgs& a, int nb) {
    using GEO = Geo<NF, 1>;
    static bool attr = false;
    if (!attr) { cudaError_t e = set_smem(hart_cols_kernel<NF>, GEO::SMEM); if (e != cudaSuccess) return (int)e; attr = true; }
    const int ntile = a.nx / 4 + 1;
    dim3 grid((ntile + GEO::G - 1) / GEO::G, nb);
    hart_cols_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_hart_cols(cudaStream_t st, int nf, const HartColsArgs& a, int nb) {
#define CALL(N) return run<N>(st, a, nb)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
