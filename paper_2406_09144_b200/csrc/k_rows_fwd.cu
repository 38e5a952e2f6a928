#include "launch.h"
namespace frs {
template <int NF, bool PAD>
static int run(cudaStream_t st, const RowsFwdArgs& a, int nb) {
    using GEO = Geo<NF, 1>;
    static bool attr = false;
    if (!attr) { cudaError_t e = set_smem(rows_fwd_kernel<NF, PAD>, GEO::SMEM); if (e != cudaSuccess) return (int)e; attr = true; }
    const int pairs = a.ny / 2;
    dim3 grid((pairs + GEO::G - 1) / GEO::G, nb);
    rows_fwd_kernel<NF, PAD><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_rows_fwd(cudaStream_t st, int nf, bool pad, const RowsFwdArgs& a, int nb) {
#define CALL(N) return pad ? run<N, true>(st, a, nb) : run<N, false>(st, a, nb)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
