#include "launch.h"
namespace frs {
template <int NF, bool PAD>
static int run(cudaStream_t st, const RowsFwdArgs& a0, int nb) {
    using GEO = typename std::conditional<PAD, RowsFwdGeo<NF>, RowsGeo<NF>>::type;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, rows_fwd_kernel<NF, PAD>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    RowsFwdArgs a = a0;
    a.items_per_batch = (a.ny / 2 + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
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
