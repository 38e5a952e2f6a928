#include "launch.h"
namespace frs {
template <int NF>
static int run(cudaStream_t st, const RowsInvArgs& a, int nb, int* grid_x) {
    using GEO = Geo<NF, 1>;
    static bool attr = false;
    if (!attr) { cudaError_t e = set_smem(rows_inv_kernel<NF>, GEO::SMEM); if (e != cudaSuccess) return (int)e; attr = true; }
    const int pairs = a.ny / 2;
    dim3 grid((pairs + GEO::G - 1) / GEO::G, nb);
    if (grid_x) *grid_x = grid.x;
    rows_inv_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_rows_inv(cudaStream_t st, int nf, const RowsInvArgs& a, int nb, int* grid_x) {
#define CALL(N) return run<N>(st, a, nb, grid_x)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
template <int NF> static int gx(int ny) { return (ny / 2 + Geo<NF, 1>::G - 1) / Geo<NF, 1>::G; }
int rows_inv_grid_x(int nf, int ny) {
#define CALL(N) return gx<N>(ny)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
