#include "launch.h"
namespace frs {
template <int NF, int MODE>
static int run(cudaStream_t st, const HartColsArgs& a0, int nb, int* grid_x) {
    using GEO = RowsGeo<NF>;
    static int cache[kMaxDevices] = {};
    int ctas = 0;
    if (int e = persistent_ctas(cache, hart_cols_kernel<NF, MODE>, GEO::THREADS, GEO::SMEM, &ctas)) return e;
    HartColsArgs a = a0;
    const int ntile = a.nx / 4 + 1;
    a.items_per_batch = (ntile + GEO::G - 1) / GEO::G;
    a.nitems = a.items_per_batch * nb;
    const int grid = a.nitems < ctas ? a.nitems : ctas;
    if (grid_x) *grid_x = grid;
    hart_cols_kernel<NF, MODE><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_hart_cols(cudaStream_t st, int nf, const HartColsArgs& a, int nb, int* grid_x) {
    // the epilogue variant follows from which optional operands are present (kernels_cols.inl HartMode)
    if (a.exp_out && (a.mul || a.add)) return (int)cudaErrorInvalidValue;
    if ((a.mul || a.add) && a.offset) return (int)cudaErrorInvalidValue;
    if (a.add && !a.mul) return (int)cudaErrorInvalidValue;
    const int mode = a.exp_out ? kHExp : !a.mul ? kHPlain : !a.add ? kHMul : !a.dot_partials ? kHMulAdd : kHMulAddDot;
#define CALL(N)                                                                         \
    switch (mode) {                                                                     \
        case kHPlain: return run<N, kHPlain>(st, a, nb, grid_x);                        \
        case kHExp: return run<N, kHExp>(st, a, nb, grid_x);                            \
        case kHMul: return run<N, kHMul>(st, a, nb, grid_x);                            \
        case kHMulAdd: return run<N, kHMulAdd>(st, a, nb, grid_x);                      \
        default: return run<N, kHMulAddDot>(st, a, nb, grid_x);                         \
    }
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}
}  // namespace frs
