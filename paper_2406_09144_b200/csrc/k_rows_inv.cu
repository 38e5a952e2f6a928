#include "launch.h"
namespace frs {
// grid_x: number of CTAs launched (= number of (sum s.c, sum j.s) partial pairs in kEnergy mode)
template <int NF, int MODE>
static int run(cudaStream_t st, const RowsInvArgs& a0, int nb, int* grid_x) {
    using GEO = RowsGeo<NF>;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, rows_inv_kernel<NF, MODE>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    RowsInvArgs a = a0;
    a.items_per_batch = (a.ny / 2 + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
    if (grid_x) *grid_x = grid;
    rows_inv_kernel<NF, MODE><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
template <int NF, int MODE>
static int run_hart(cudaStream_t st, const RowsInvHartArgs& a0, int nb, int* grid_x) {
    using GEO = RowsInvHartGeo<NF>;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, rows_inv_hart_kernel<NF, MODE>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    RowsInvHartArgs a = a0;
    a.inv.items_per_batch = (a.inv.ny / 2 + GEO::G - 1) / GEO::G;
    a.inv.nitems = a.inv.items_per_batch * nb;
    const int grid = a.inv.nitems < ctas ? a.inv.nitems : ctas;
    if (grid_x) *grid_x = grid;
    rows_inv_hart_kernel<NF, MODE><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_rows_inv_hart(cudaStream_t st, int nf, const RowsInvHartArgs& a, int nb, int* grid_x) {
#define CALLH(N) return a.inv.mode == kMulS ? run_hart<N, kMulS>(st, a, nb, grid_x) : run_hart<N, kEnergy>(st, a, nb, grid_x)
    switch (nf) {
        case 1024: CALLH(1024);
        case 2048: CALLH(2048);
        case 4096: CALLH(4096);
        default: return (int)cudaErrorInvalidValue;
    }
#undef CALLH
}
int launch_rows_inv(cudaStream_t st, int nf, const RowsInvArgs& a, int nb, int* grid_x) {
#define CALL(N)                                                            \
    return a.mode == kPlain ? run<N, kPlain>(st, a, nb, grid_x)            \
         : a.mode == kMulS  ? run<N, kMulS>(st, a, nb, grid_x)             \
         : a.mode == kResid ? run<N, kResid>(st, a, nb, grid_x)            \
                            : run<N, kEnergy>(st, a, nb, grid_x)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
