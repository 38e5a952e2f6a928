#include "launch.h"
namespace frs {
template <int NF>
static int run(cudaStream_t st, const HartColsArgs& a0, int nb, int* grid_x) {
    using GEO = RowsGeo<NF>;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, hart_cols_kernel<NF>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    HartColsArgs a = a0;
    const int ntile = a.nx / 4 + 1;
    a.items_per_batch = (ntile + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
    if (grid_x) *grid_x = grid;
    hart_cols_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_hart_cols(cudaStream_t st, int nf, const HartColsArgs& a, int nb, int* grid_x) {
#define CALL(N) return run<N>(st, a, nb, grid_x)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
