// frs_api.cu -- the C ABI of include/frs.h: context, setup, and the launch sequences of the hot
// path.  Every step of the path runs in the kernels of this library;
// there is no CPU fallback: without a CUDA device frs_create fails with FRS_ECUDA.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <vector>

#include "../../include/frs.h"
#include "ew_kernels.cuh"
#include "launch.h"
#include "prior.h"
#include "response.h"
#include "setup.h"
#include "tables.h"

using namespace frs;

namespace {
enum PassKind { kPassRowsFwd = 0, kPassConvCols = 1, kPassRowsInv = 2, kPassHartRows = 3, kPassHartCols = 4, kNPass = 5 };
struct ProfRec { int kind; cudaEvent_t a, b; };
constexpr int kMaxRedBlocks = 1184;   // 148 SMs x 8
constexpr size_t kMaxProfRecords = 4096;
}  // namespace

struct frs_ctx {
    int ny = 0, nx = 0, nchan = 0, nfield = 0, device = 0;
    cudaStream_t stream = nullptr;
    size_t npix = 0;
    int ntile = 0, ntile_h = 0;
    std::map<int, float4*> tw;       // stage twiddles of the sorting core, per transform length
    std::map<int, float4*> twd;      // twiddles of the DIF/DIT core (column convolution, length >= 256)
    std::map<int, float2*> twist;
    // two orientations of the sky-space arrays: natural [ny][nx] (public sky-space calls) and
    // transposed [nx][ny] (latent-space path: each 2-pass Hartley transform transposes for free)
    float *wt = nullptr, *wtT = nullptr, *dirty = nullptr, *dirtyT = nullptr, *amp = nullptr, *s = nullptr, *sT = nullptr;
    bool s_ok = false, sT_ok = false;
    float *d_mu = nullptr, *d_lognu = nullptr;
    float2 *T = nullptr, *T2 = nullptr, *Th = nullptr;   // T: block layout (rows_fwd -> conv_cols); T2: columns (conv_cols -> rows_inv)
    struct MapKey { const void* p; int rows, nf, nb; CUtensorMap row, col; };   // col: of T; row: columns map of T2
    std::vector<MapKey> maps;  // spectrum tensor maps (tmap.h), built on first use
    float *lin = nullptr, *img = nullptr, *acc = nullptr;
    // Eq. 9 with the fitted noise kernel (R14): K, 1/(K ny nx) in both orientations, two more image-sized scratch arrays
    float *kern = nullptr, *kinvN = nullptr, *kinvT = nullptr, *kisqN = nullptr, *img2 = nullptr, *img3 = nullptr;
    float *lat1 = nullptr, *lat2 = nullptr;
    float* visbuf = nullptr; size_t visbuf_n = 0;   // visibilities of the exact response (major cycle)   // latent-sized scratch of the MGVI calls (sample source, positions xi +- sigma)
    bool have_kern = false;
    int lik_mode = 0;                // 0: N' = R' limit, 1: Eq. 9 with N'^-1 of Eq. 18
    float *cg_r = nullptr, *cg_p = nullptr, *cg_q = nullptr;
    float *hx = nullptr, *hy = nullptr, *hx2 = nullptr, *hy2 = nullptr;
    cudaStream_t s_in = nullptr, s_out = nullptr;      // copy streams of frs_sky_metric_apply_host_batch
    cudaEvent_t ev_in[2] = {}, ev_comp[2] = {}, ev_out[2] = {};
    double *partials = nullptr, *scal = nullptr;   // scal: [0..7] CG, [8] sum s.c, [9] sum j.s, [10] <xi,xi>, [11] E
    int* flag = nullptr;
    bool guard = false;                // FRS_GUARD=1: guard zones around every ctx-owned array
    struct Guard { char* base; size_t used, padded; };
    std::vector<Guard> guards;
    bool have_psf = false, have_dirty = false, have_amp = false, have_s = false;
    long long launches = 0;
    // one CG iteration captured as a CUDA graph (cg_solve_impl): replayed while the key (every frozen argument) matches
    struct CgGraphKey { const float* x; int with_prior, nfield, lik_mode; double* hist; double rtol2; bool sT_ok, pts_in_sky; long long epoch; } cg_key = {};
    long long cfg_epoch = 0;           // bumped by every setter that can change the launch sequence of an iteration
    cudaGraphExec_t cg_exec = nullptr;
    cudaStream_t cap_stream = nullptr;  // capture runs on a stream of the ctx's own (the caller's may be the legacy default stream)
    long long cg_graph_launches = 0;   // kernels per replay
    int use_graphs = 1;
    int fuse_inv_hart = 1;             // latent-space path: rows_inv and the following Hartley row pass as one kernel
    // NEXT-3: learned amplitude spectrum (prior.h).  plain_latent: the joint calls run the latent-space passes without
    // the fused (.A, + v) prologue / epilogue and apply their own
    AmpModel am;
    bool have_amp_model = false, plain_latent = false;
    // inverse-gamma point-source pixels (reading R18): fluxes added to the cached sky; the latent-space passes patch the
    // few pixels where the Jacobian of the diffuse part differs from the total sky (points_pre / points_post)
    PointSources pts;
    std::vector<int> pts_yx;            // host copy of the point pixels (y, x), re-validated when the field of view changes
    int fov_y = 0, fov_x = 0;           // image smaller than the grid (reading R19): the sky is zero outside [0,fov_y) x [0,fov_x); 0 = whole grid
    const float* pts_dv = nullptr;      // tangent of the point latents (joint metric), else null = 0
    const float* pts_add = nullptr;     // prior term added to the point outputs (joint calls with the prior), else null
    float* pts_out = nullptr;           // where the point outputs go (joint calls), else the scratch pts.out
    bool profiling = false;
    std::vector<ProfRec> prof;
    char err[512] = "no error";
};

namespace {

int fail(frs_ctx* c, int code, const char* msg) {
    if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
    return code;
}
int cuda_fail(frs_ctx* c, cudaError_t e, const char* where) {
    if (c) snprintf(c->err, sizeof(c->err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
    return FRS_ECUDA;
}
#define CK(call)                                                          \
    do {                                                                  \
        cudaError_t e_ = (call);                                          \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);          \
    } while (0)
#define CKL(call)                                                         \
    do {                                                                  \
        int e_ = (call);                                                  \
        if (e_ != 0) return cuda_fail(ctx, (cudaError_t)e_, #call);       \
    } while (0)
#define RET(call)                     \
    do {                              \
        int r_ = (call);              \
        if (r_ != FRS_OK) return r_;  \
    } while (0)

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
bool pow2_in(int n, int lo, int hi) { return n >= lo && n <= hi && (n & (n - 1)) == 0; }

struct Prof {
    frs_ctx* c; int kind; cudaEvent_t a = nullptr, b = nullptr;
    Prof(frs_ctx* c_, int kind_) : c(c_), kind(kind_) {
        // at most kMaxProfRecords pending records (events are released by frs_profile_read): later passes go untimed
        if (c->profiling && c->prof.size() < kMaxProfRecords) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, c->stream); }
    }
    ~Prof() {
        if (!a) return;
        cudaEventRecord(b, c->stream);
        c->prof.push_back({kind, a, b});
    }
};

// Guard zones (debug; the environment variable FRS_GUARD=1 at frs_create): every ctx-owned array gets kGuardBytes of a
// byte pattern in front of and behind it, and frs_debug_check_guards counts the arrays whose pattern was touched -- the
// stand-in for compute-sanitizer memcheck, which is closed on the GPU pool (profiles/r2_sanitizer.md).
constexpr size_t kGuardBytes = 4096;
constexpr int kGuardByte = 0xA5;
template <typename T>
int dev_alloc(frs_ctx* ctx, T** p, size_t count) {
    if (*p) return FRS_OK;
    if (!ctx->guard) {
        CK(cudaMalloc(reinterpret_cast<void**>(p), count * sizeof(T)));
        return FRS_OK;
    }
    const size_t bytes = (count * sizeof(T) + 255) & ~(size_t)255;
    char* base = nullptr;
    CK(cudaMalloc(reinterpret_cast<void**>(&base), bytes + 2 * kGuardBytes));
    CK(cudaMemset(base, kGuardByte, kGuardBytes));
    CK(cudaMemset(base + kGuardBytes + count * sizeof(T), kGuardByte, bytes - count * sizeof(T) + kGuardBytes));
    *p = reinterpret_cast<T*>(base + kGuardBytes);
    ctx->guards.push_back({base, count * sizeof(T), bytes});
    return FRS_OK;
}
void dev_free(frs_ctx* ctx, void* p) {
    if (!p) return;
    for (auto& g : ctx->guards)
        if (g.base + kGuardBytes == p) { cudaFree(g.base); g.base = nullptr; return; }
    cudaFree(p);
}

int ensure_tables(frs_ctx* ctx, int n) {
    if (ctx->tw.count(n)) return FRS_OK;
    std::vector<float4> tw = build_twiddles(n);
    std::vector<float2> ts = build_twist(n);
    float4* dtw = nullptr;
    float2* dts = nullptr;
    CK(cudaMalloc(reinterpret_cast<void**>(&dtw), tw.size() * sizeof(float4)));
    CK(cudaMalloc(reinterpret_cast<void**>(&dts), ts.size() * sizeof(float2)));
    CK(cudaMemcpy(dtw, tw.data(), tw.size() * sizeof(float4), cudaMemcpyHostToDevice));
    CK(cudaMemcpy(dts, ts.data(), ts.size() * sizeof(float2), cudaMemcpyHostToDevice));
    ctx->tw[n] = dtw;
    ctx->twist[n] = dts;
    if (conv_cols_uses_dif(n)) {
        std::vector<float4> td = build_dif_twiddles(n);
        float4* dtd = nullptr;
        CK(cudaMalloc(reinterpret_cast<void**>(&dtd), td.size() * sizeof(float4)));
        CK(cudaMemcpy(dtd, td.data(), td.size() * sizeof(float4), cudaMemcpyHostToDevice));
        ctx->twd[n] = dtd;
    }
    return FRS_OK;
}

size_t max2(size_t a, size_t b) { return a > b ? a : b; }

int ensure_scratch(frs_ctx* ctx) {
    const size_t np = ctx->npix, ny = ctx->ny, nx = ctx->nx;
    RET(dev_alloc(ctx, &ctx->T, (size_t)ctx->nchan * max2(spec_batch_stride(ctx->ny, ctx->nx), spec_batch_stride(ctx->nx, ctx->ny))));
    RET(dev_alloc(ctx, &ctx->T2, (size_t)ctx->nchan * max2((nx / 2 + 1) * ny, (ny / 2 + 1) * nx) * 2));
    RET(dev_alloc(ctx, &ctx->Th, (size_t)(ctx->nchan > 2 ? ctx->nchan : 2) *
                                     max2(spec_batch_stride(ctx->ny, ctx->nx / 2, kPairBins), spec_batch_stride(ctx->nx, ctx->ny / 2, kPairBins))));
    RET(dev_alloc(ctx, &ctx->lin, 2 * np));
    RET(dev_alloc(ctx, &ctx->acc, 2 * np));
    RET(dev_alloc(ctx, &ctx->img, (size_t)ctx->nchan * np));
    RET(dev_alloc(ctx, &ctx->s, (size_t)ctx->nchan * np));
    RET(dev_alloc(ctx, &ctx->sT, (size_t)ctx->nchan * np));
    return FRS_OK;
}

int red_blocks(size_t n) {
    size_t b = (n / 4 + kRedThreads - 1) / kRedThreads;
    return (int)(b < 1 ? 1 : (b > (size_t)kMaxRedBlocks ? kMaxRedBlocks : b));
}

// out = sum a.b  -> device double
int dot(frs_ctx* ctx, const float* a, const float* b, size_t n, double* d_out) {
    const int nb = red_blocks(n);
    dot_partial_kernel<<<nb, kRedThreads, 0, ctx->stream>>>(a, b, n, ctx->partials);
    reduce_final_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->partials, nb, 1, 0, d_out);
    ctx->launches += 2;
    CK(cudaGetLastError());
    return FRS_OK;
}

// ---- the three passes of C (Eq. 14) -----------------------------------------------------------
// Orientation of a sky-space image: [rows][len].  Natural: rows = ny, len = nx.  Transposed: rows = nx,
// len = ny, with the weight table built for the transposed PSF spectrum.
struct Orient { int rows, len, ntile; const float* wt; };
Orient orient(const frs_ctx* ctx, bool transposed) {
    return transposed ? Orient{ctx->nx, ctx->ny, ctx->ny / 2 + 1, ctx->wtT} : Orient{ctx->ny, ctx->nx, ctx->nx / 2 + 1, ctx->wt};
}
// tensor maps of a spectrum buffer in the block layout (tmap.h), cached per shape
int spectrum_maps(frs_ctx* ctx, const float2* T, int rows, int nf, int nb, CUtensorMap* row, CUtensorMap* col) {
    for (const auto& k : ctx->maps)
        if (k.p == T && k.rows == rows && k.nf == nf && k.nb == nb) {
            if (row) *row = k.row;
            if (col) *col = k.col;
            return FRS_OK;
        }
    frs_ctx::MapKey k{T, rows, nf, nb, {}, {}};
    if (make_spectrum_col_map(&k.col, T, rows, nf, nb) || make_columns_map(&k.row, ctx->T2, rows, nf, nf + 2, nb))
        return fail(ctx, FRS_ECUDA, "cuTensorMapEncodeTiled failed");
    ctx->maps.push_back(k);
    if (row) *row = k.row;
    if (col) *col = k.col;
    return FRS_OK;
}

int conv_rows_fwd(frs_ctx* ctx, const Orient& o, const float* in, const float* mul) {
    Prof pr(ctx, kPassRowsFwd);
    RowsFwdArgs a{};
    a.in = in; a.mul = mul; a.out = ctx->T; a.ny = o.rows;
    a.in_bstride = ctx->npix; a.mul_bstride = ctx->npix;
    a.scale = 1.0f;   // yields 2 X[k]; the 1/2 is folded into wt
    a.tw = ctx->tw[o.len]; a.twist = ctx->twist[o.len];
    CKL(launch_rows_fwd(ctx->stream, o.len, true, a, ctx->nchan));
    ctx->launches++;
    return FRS_OK;
}
int conv_cols(frs_ctx* ctx, const Orient& o) {
    Prof pr(ctx, kPassConvCols);
    ConvColsArgs a{};
    a.t = ctx->T; a.out = ctx->T2; a.wt = o.wt; a.ncols = o.len + 1; a.ntile = o.ntile;
    RET(spectrum_maps(ctx, ctx->T, o.rows, o.len, ctx->nchan, nullptr, &a.tmap));
    a.w_bstride = (size_t)o.ntile * 2 * o.rows * 2;
    a.tw = conv_cols_uses_dif(o.rows) ? ctx->twd[o.rows] : ctx->tw[o.rows];
    a.twist = ctx->twist[o.rows];
    CKL(launch_conv_cols(ctx->stream, o.rows, a, ctx->nchan));
    ctx->launches++;
    return FRS_OK;
}
int conv_rows_inv(frs_ctx* ctx, const Orient& o, float* out, int mode, const float* s, const float* j, int* grid_x) {
    Prof pr(ctx, kPassRowsInv);
    RowsInvArgs a{};
    a.t = ctx->T2; a.out = out; a.s = s; a.j = j; a.partials = ctx->partials;
    a.ny = o.rows; a.mode = mode; a.cols = 2 * o.ntile;
    RET(spectrum_maps(ctx, ctx->T, o.rows, o.len, ctx->nchan, &a.tmap, nullptr));
    a.img_bstride = ctx->npix;
    a.tw = ctx->tw[o.len]; a.twist = ctx->twist[o.len];
    CKL(launch_rows_inv(ctx->stream, o.len, a, ctx->nchan, grid_x));
    ctx->launches++;
    return FRS_OK;
}

// TRANSPOSING 2-D Hartley transform, two passes:  in [nb][n1][n2]  ->  out [nb][n2][n1],
//   out[x][y] = (mul[x][y] .) ( H[premul . in][y][x] + offset[b] ) (+ add[x][y]).
// The row pass leaves column tiles, and the column pass of column x produces H[.][x] for all y, which is
// one contiguous run of the transposed output -- so the transform transposes for free, and the
// latent-space path keeps its sky-space arrays transposed instead of paying for scattered stores.
// second half of hartley_t: the column pass over ctx->Th
int hartley_cols(frs_ctx* ctx, int n1, int n2, float* out, const float* mul, const float* add, const float* offset_dev, int nb,
                 double* d_dot = nullptr, bool exp_out = false) {
    Prof pr(ctx, kPassHartCols);
    HartColsArgs a{};
    a.t = ctx->Th; a.out = out; a.mul = mul; a.add = add; a.offset = offset_dev; a.nx = n2; a.exp_out = exp_out ? 1 : 0;
    a.img_bstride = ctx->npix;
    a.tw = ctx->tw[n1];
    a.dot_partials = (d_dot && add) ? ctx->partials : nullptr;   // <add, out> fused into the epilogue (fp64)
    int gx = 0;
    CKL(launch_hart_cols(ctx->stream, n1, a, nb, &gx));
    ctx->launches++;
    if (a.dot_partials) {
        reduce_final_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->partials, gx, 1, 0, d_dot);
        ctx->launches++;
    }
    return FRS_OK;
}
int hartley_t(frs_ctx* ctx, const float* in, int n1, int n2, const float* premul, float* out, const float* mul,
              const float* add, const float* offset_dev, int nb, double* d_dot = nullptr, float sign = 1.0f,
              bool exp_out = false) {
    {
        Prof pr(ctx, kPassHartRows);
        RowsFwdArgs a{};
        a.in = in; a.mul = premul; a.out = ctx->Th; a.ny = n1;
        a.in_bstride = ctx->npix; a.mul_bstride = ctx->npix;
        a.scale = 0.5f * sign;   // sign = -1: the transform of -in (offset must be absent)
        a.tw = ctx->tw[n2 / 2]; a.twist = ctx->twist[n2 / 2];
        CKL(launch_rows_fwd(ctx->stream, n2 / 2, false, a, nb));
        ctx->launches++;
    }
    return hartley_cols(ctx, n1, n2, out, mul, add, offset_dev, nb, d_dot, exp_out);
}

// The inverse row pass of the convolution fused with the row pass of the Hartley transform of its result
// (kernels_inv_hart.inl): T2 -> Th without the image in between.  mode: kMulS or kEnergy.  Follow with hartley_cols.
bool fused_inv_hart_ok(const frs_ctx* ctx, const Orient& o) {
    return ctx->fuse_inv_hart && rows_inv_hart_ok(o.len) && ctx->nchan == 1 && ctx->nfield == 1 && !ctx->profiling &&
           !(ctx->pts.n > 0 && ctx->pts.in_sky);
}
int conv_rows_inv_hart(frs_ctx* ctx, const Orient& o, int mode, const float* s, const float* j, float sign, int* grid_x) {
    RowsInvHartArgs h{};
    RowsInvArgs& a = h.inv;
    a.t = ctx->T2; a.out = nullptr; a.s = s; a.j = j; a.partials = ctx->partials;
    a.ny = o.rows; a.mode = mode; a.cols = 2 * o.ntile;
    RET(spectrum_maps(ctx, ctx->T, o.rows, o.len, ctx->nchan, &a.tmap, nullptr));
    a.img_bstride = ctx->npix;
    a.tw = ctx->tw[o.len]; a.twist = ctx->twist[o.len];
    h.th = ctx->Th; h.scale = 0.5f * sign;
    h.tw2 = ctx->tw[o.len / 2]; h.twist2 = ctx->twist[o.len / 2];
    CKL(launch_rows_inv_hart(ctx->stream, o.len, h, ctx->nchan, grid_x));
    ctx->launches++;
    return FRS_OK;
}

int transpose(frs_ctx* ctx, const float* in, float* out, int rows, int cols, int nb) {
    CKL(launch_transpose(ctx->stream, in, out, rows, cols, nb));
    ctx->launches++;
    return FRS_OK;
}
int need_s_natural(frs_ctx* ctx) {
    if (!ctx->s_ok) { RET(transpose(ctx, ctx->sT, ctx->s, ctx->nx, ctx->ny, ctx->nchan)); ctx->s_ok = true; }
    return FRS_OK;
}
int need_s_transposed(frs_ctx* ctx) {
    if (!ctx->sT_ok) { RET(transpose(ctx, ctx->s, ctx->sT, ctx->ny, ctx->nx, ctx->nchan)); ctx->sT_ok = true; }
    return FRS_OK;
}

int ew_grid(size_t npix) { return (int)((npix / 4 + kEwThreads - 1) / kEwThreads); }

int check_hot(frs_ctx* ctx, bool need_s, bool need_model) {
    if (!ctx) return FRS_EINVAL;
    if (!ctx->have_psf) return fail(ctx, FRS_ESTATE, "PSF not set (frs_set_psf / frs_set_psf_weights)");
    if (need_model && !ctx->have_amp) return fail(ctx, FRS_ESTATE, "amplitude spectrum not set (frs_set_amplitude)");
    if (need_s && !ctx->have_s) return fail(ctx, FRS_ESTATE, "no position set (frs_sky_forward / frs_energy_grad / frs_set_sky)");
    return ensure_scratch(ctx);
}

int sky_forward_impl(frs_ctx* ctx, const float* xi) {
    // tau_f = mu_f + H[A_f xi_f];  s_c = exp(tau_0 + lognu_c tau_1)      (R6)   -- sky-space arrays transposed
    if (ctx->nfield == 1 && ctx->nchan == 1) {
        // single field, single channel: s = exp(tau) leaves the last Hartley pass directly (A2 fused into A1)
        RET(hartley_t(ctx, xi, ctx->ny, ctx->nx, ctx->amp, ctx->sT, nullptr, nullptr, ctx->d_mu, 1, nullptr, 1.0f, true));
    } else {
        RET(hartley_t(ctx, xi, ctx->ny, ctx->nx, ctx->amp, ctx->lin, nullptr, nullptr, ctx->d_mu, ctx->nfield));
        sky_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->lin, ctx->d_lognu, ctx->sT, ctx->npix, ctx->nfield, ctx->nchan);
        ctx->launches++;
    }
    CK(cudaGetLastError());
    if (ctx->pts.n > 0) {
        CKL(launch_points_flux(ctx->stream, ctx->pts));
        CKL(launch_points_add(ctx->stream, ctx->pts, ctx->sT));
        ctx->launches += 2;
        ctx->pts.in_sky = true;
    }
    if (ctx->fov_y) {                        // sT is [nx][ny]
        CKL(launch_mask_outside(ctx->stream, ctx->sT, ctx->nx, ctx->ny, ctx->fov_x, ctx->fov_y, ctx->nchan));
        ctx->launches++;
    }
    ctx->have_s = true;
    ctx->sT_ok = true;
    ctx->s_ok = false;
    return FRS_OK;
}

// point-source pixels around the fused . s passes (no-ops without point sources in the cached sky)
int points_pre(frs_ctx* ctx, float* lin) {
    if (ctx->pts.n > 0 && ctx->pts.in_sky) {
        CKL(launch_points_pre(ctx->stream, ctx->pts, lin, ctx->pts_dv));
        ctx->launches++;
    }
    return FRS_OK;
}
int points_post(frs_ctx* ctx, float* acc, double sign, double* energy_acc) {
    if (ctx->pts.n > 0 && ctx->pts.in_sky) {
        CKL(launch_points_post(ctx->stream, ctx->pts, acc, ctx->pts_add, ctx->pts_out ? ctx->pts_out : ctx->pts.out, sign,
                               ctx->pts_add ? energy_acc : nullptr));
        ctx->launches++;
    }
    return FRS_OK;
}

// ---- Eq. 9 with the fitted noise kernel (reading R14) -------------------------------------
// u = N'^-1 r = H[ K^-1 . H[r] ] / (ny nx) for the real even kernel K (Eq. 18: periodic, unpadded), in the transposed
// orientation of the latent-space path: r, u [nchan][nx][ny]; the intermediate is in the natural orientation.
int ninv_transposed(frs_ctx* ctx, const float* r, float* u) {
    RET(hartley_t(ctx, r, ctx->nx, ctx->ny, nullptr, ctx->img3, ctx->kinvN, nullptr, nullptr, ctx->nchan));
    RET(hartley_t(ctx, ctx->img3, ctx->ny, ctx->nx, nullptr, u, nullptr, nullptr, nullptr, ctx->nchan));
    return FRS_OK;
}
int ensure_scratch9(frs_ctx* ctx) {
    RET(dev_alloc(ctx, &ctx->img2, (size_t)ctx->nchan * ctx->npix));
    RET(dev_alloc(ctx, &ctx->img3, (size_t)ctx->nchan * ctx->npix));
    return FRS_OK;
}

// M v = J^T C N'^-1 C J v (+ v): three convolutions per apply (two padded, one periodic)
int metric_apply9_impl(frs_ctx* ctx, const float* v, int with_prior, float* out, double* d_vmv) {
    const Orient o = orient(ctx, true);
    RET(need_s_transposed(ctx));
    RET(ensure_scratch9(ctx));
    RET(hartley_t(ctx, v, ctx->ny, ctx->nx, ctx->plain_latent ? nullptr : ctx->amp, ctx->lin, nullptr, nullptr, nullptr, ctx->nfield));
    const bool simple = ctx->nchan == 1 && ctx->nfield == 1;
    if (simple) {
        RET(points_pre(ctx, ctx->lin));
        RET(conv_rows_fwd(ctx, o, ctx->lin, ctx->sT));
    } else {
        jvp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->lin, ctx->sT, ctx->d_lognu, ctx->img,
                                                                               ctx->npix, ctx->nfield, ctx->nchan);
        ctx->launches++;
        RET(conv_rows_fwd(ctx, o, ctx->img, nullptr));
    }
    RET(conv_cols(ctx, o));
    RET(conv_rows_inv(ctx, o, ctx->img2, kPlain, nullptr, nullptr, nullptr));            // C J v
    RET(ninv_transposed(ctx, ctx->img2, ctx->img));                                       // N'^-1 C J v
    RET(conv_rows_fwd(ctx, o, ctx->img, nullptr));
    RET(conv_cols(ctx, o));
    if (simple && fused_inv_hart_ok(ctx, o)) {
        RET(conv_rows_inv_hart(ctx, o, kMulS, ctx->sT, nullptr, 1.0f, nullptr));
        RET(hartley_cols(ctx, ctx->nx, ctx->ny, out, ctx->plain_latent ? nullptr : ctx->amp,
                         (with_prior && !ctx->plain_latent) ? v : nullptr, nullptr, ctx->nfield,
                         (with_prior && !ctx->plain_latent) ? d_vmv : nullptr));
        CK(cudaGetLastError());
        return FRS_OK;
    }
    if (simple) {
        RET(conv_rows_inv(ctx, o, ctx->acc, kMulS, ctx->sT, nullptr, nullptr));
        RET(points_post(ctx, ctx->acc, 1.0, nullptr));
    } else {
        RET(conv_rows_inv(ctx, o, ctx->img, kMulS, ctx->sT, nullptr, nullptr));
        vjp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->img, ctx->d_lognu, ctx->acc, ctx->npix,
                                                                               ctx->nfield, ctx->nchan);
        ctx->launches++;
    }
    RET(hartley_t(ctx, ctx->acc, ctx->nx, ctx->ny, nullptr, out, ctx->plain_latent ? nullptr : ctx->amp,
                  (with_prior && !ctx->plain_latent) ? v : nullptr, nullptr, ctx->nfield,
                  (with_prior && !ctx->plain_latent) ? d_vmv : nullptr));
    CK(cudaGetLastError());
    return FRS_OK;
}

// d_vmv (device, optional, needs with_prior): <v, M v>, accumulated in the last pass instead of a separate dot
int metric_apply_impl(frs_ctx* ctx, const float* v, int with_prior, float* out, double* d_vmv = nullptr) {
    if (ctx->lik_mode == 1) return metric_apply9_impl(ctx, v, with_prior, out, d_vmv);
    const Orient o = orient(ctx, true);
    RET(need_s_transposed(ctx));
    // lin_f = H[A_f v_f]   (transposed)
    RET(hartley_t(ctx, v, ctx->ny, ctx->nx, ctx->plain_latent ? nullptr : ctx->amp, ctx->lin, nullptr, nullptr, nullptr, ctx->nfield));
    const bool simple = ctx->nchan == 1 && ctx->nfield == 1;
    if (simple) {
        RET(points_pre(ctx, ctx->lin));
        RET(conv_rows_fwd(ctx, o, ctx->lin, ctx->sT));             // s . lin fused into the row pass
    } else {
        jvp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->lin, ctx->sT, ctx->d_lognu, ctx->img,
                                                                               ctx->npix, ctx->nfield, ctx->nchan);
        ctx->launches++;
        RET(conv_rows_fwd(ctx, o, ctx->img, nullptr));
    }
    RET(conv_cols(ctx, o));
    if (simple && fused_inv_hart_ok(ctx, o)) {
        // acc = s . C(...) never reaches memory: its rows go straight into the row pass of the transform below
        RET(conv_rows_inv_hart(ctx, o, kMulS, ctx->sT, nullptr, 1.0f, nullptr));
        RET(hartley_cols(ctx, ctx->nx, ctx->ny, out, ctx->plain_latent ? nullptr : ctx->amp,
                         (with_prior && !ctx->plain_latent) ? v : nullptr, nullptr, ctx->nfield,
                         (with_prior && !ctx->plain_latent) ? d_vmv : nullptr));
        CK(cudaGetLastError());
        return FRS_OK;
    }
    if (simple) {
        RET(conv_rows_inv(ctx, o, ctx->acc, kMulS, ctx->sT, nullptr, nullptr));      // acc = s . C(...)
        RET(points_post(ctx, ctx->acc, 1.0, nullptr));
    } else {
        RET(conv_rows_inv(ctx, o, ctx->img, kMulS, ctx->sT, nullptr, nullptr));
        vjp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->img, ctx->d_lognu, ctx->acc, ctx->npix,
                                                                               ctx->nfield, ctx->nchan);
        ctx->launches++;
    }
    // out_f = A_f . H[acc_f] (+ v_f)   (transposes back to the latent layout)
    RET(hartley_t(ctx, ctx->acc, ctx->nx, ctx->ny, nullptr, out, ctx->plain_latent ? nullptr : ctx->amp,
                  (with_prior && !ctx->plain_latent) ? v : nullptr, nullptr, ctx->nfield,
                  (with_prior && !ctx->plain_latent) ? d_vmv : nullptr));
    CK(cudaGetLastError());
    return FRS_OK;
}

int cg_alloc(frs_ctx* ctx) {
    RET(dev_alloc(ctx, &ctx->cg_r, 2 * ctx->npix));     // sized for two fields whatever nfield is now
    RET(dev_alloc(ctx, &ctx->cg_p, 2 * ctx->npix));
    RET(dev_alloc(ctx, &ctx->cg_q, 2 * ctx->npix));
    return FRS_OK;
}

// second half of an iteration: from q = M p to the updated (x, r, p, scal)
int cg_iter_finish(frs_ctx* ctx, float* x, double* d_hist, int k, bool have_pq = false, double rtol2 = 0.0) {
    const size_t n = (size_t)ctx->nfield * ctx->npix;
    const int nb = red_blocks(n);
    if (!have_pq) RET(dot(ctx, ctx->cg_p, ctx->cg_q, n, ctx->scal + kPQ));
    cg_update_xr_kernel<<<nb, kRedThreads, 0, ctx->stream>>>(x, ctx->cg_r, ctx->cg_p, ctx->cg_q, n, ctx->scal, ctx->partials);
    reduce_final_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->partials, nb, 1, 0, ctx->scal + kRRNew);
    cg_update_p_kernel<<<nb, kEwThreads, 0, ctx->stream>>>(ctx->cg_p, ctx->cg_r, n, ctx->scal, ctx->scal + kBeta);
    cg_shift_kernel<<<1, 1, 0, ctx->stream>>>(ctx->scal, d_hist, k < 0 ? -1 : k + 1, rtol2);
    ctx->launches += 4;
    CK(cudaGetLastError());
    return FRS_OK;
}
// one iteration from (x, r, p, scal[kRR]); leaves scal[kRR] = new <r,r>
int cg_iter(frs_ctx* ctx, float* x, int with_prior, double* d_hist, int k, double rtol2 = 0.0) {
    // with the prior term the last Hartley pass has p and q = M p side by side: <p, q> comes out of its epilogue
    RET(metric_apply_impl(ctx, ctx->cg_p, with_prior, ctx->cg_q, with_prior ? ctx->scal + kPQ : nullptr));
    return cg_iter_finish(ctx, x, d_hist, k, with_prior != 0, rtol2);
}

float* ctx_lat1(frs_ctx* ctx) { return ctx->lat1; }

// positions xi + sigma_i (and xi - sigma_i): visit(position, weight, first)
template <typename F>
int for_each_position(frs_ctx* ctx, const float* xi, const float* samples, int ns, int mirrored, F visit) {
    const size_t n = (size_t)ctx->nfield * ctx->npix;
    const int npos = ns * (mirrored ? 2 : 1);
    int k = 0;
    for (int i = 0; i < ns; ++i)
        for (int sgn = 1; sgn >= (mirrored ? -1 : 1); sgn -= 2, ++k) {
            add_scaled_kernel<<<ew_grid(n), kEwThreads, 0, ctx->stream>>>(xi, samples + (size_t)i * n, (float)sgn, ctx_lat1(ctx), n);
            ctx->launches++;
            RET(visit(ctx_lat1(ctx), 1.0f / (float)npos, k == 0));
        }
    return FRS_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

#define FRS_STR_(x) #x
#define FRS_STR(x) FRS_STR_(x)
const char* frs_version(void) {
    return "frs 0.3 (sm_100a; packed-pair register FFT passes: sorting core for the row and Hartley passes, DIF/DIT core for the column convolution)"
#if defined(FRS_STRIP) && FRS_STRIP != 0
           " ATTRIBUTION BUILD FRS_STRIP=" FRS_STR(FRS_STRIP) ": conv_cols_dif results are wrong by construction"
#endif
        ;
}

const char* frs_last_error(const frs_ctx* ctx) { return ctx ? ctx->err : "null context"; }

long long frs_launch_count(const frs_ctx* ctx) { return ctx ? ctx->launches : 0; }

int frs_create(int ny, int nx, int nchan, int device, void* stream, frs_ctx** out) {
    if (!out) return FRS_EINVAL;
    *out = nullptr;
    if (!pow2_in(ny, 32, 4096) || !pow2_in(nx, 32, 4096) || nchan < 1) return FRS_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return FRS_ECUDA;
    if (cudaSetDevice(device) != cudaSuccess) return FRS_ECUDA;
    frs_ctx* ctx = new frs_ctx();
    ctx->ny = ny; ctx->nx = nx; ctx->nchan = nchan; ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(stream);
    { const char* e = getenv("FRS_GUARD"); ctx->guard = e && e[0] == '1'; }
    ctx->npix = (size_t)ny * nx;
    ctx->ntile = nx / 2 + 1;
    ctx->ntile_h = nx / 4 + 1;
    int rc = FRS_OK;
    auto init = [&]() -> int {
        RET(ensure_tables(ctx, nx));
        RET(ensure_tables(ctx, ny));
        RET(ensure_tables(ctx, nx / 2));
        RET(ensure_tables(ctx, ny / 2));
        RET(dev_alloc(ctx, &ctx->partials, (size_t)1 << 16));
        RET(dev_alloc(ctx, &ctx->scal, 16));
        RET(dev_alloc(ctx, &ctx->flag, 4));
        RET(dev_alloc(ctx, &ctx->d_mu, 2));
        RET(dev_alloc(ctx, &ctx->d_lognu, (size_t)nchan));
        CK(cudaMemset(ctx->scal, 0, 16 * sizeof(double)));
        CK(cudaMemset(ctx->d_mu, 0, 2 * sizeof(float)));
        CK(cudaMemset(ctx->d_lognu, 0, nchan * sizeof(float)));
        return FRS_OK;
    };
    rc = init();
    if (rc != FRS_OK) { frs_destroy(ctx); return rc; }
    *out = ctx;
    return FRS_OK;
}

void frs_destroy(frs_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto& kv : ctx->tw) cudaFree(kv.second);
    for (auto& kv : ctx->twd) cudaFree(kv.second);
    for (auto& kv : ctx->twist) cudaFree(kv.second);
    void* ptrs[] = {ctx->visbuf, ctx->kern, ctx->kinvN, ctx->kinvT, ctx->kisqN, ctx->lat1, ctx->lat2, ctx->img2, ctx->img3, ctx->wt, ctx->wtT, ctx->dirty, ctx->dirtyT, ctx->amp, ctx->s, ctx->sT, ctx->d_mu, ctx->d_lognu, ctx->T, ctx->T2, ctx->Th, ctx->lin, ctx->img,
                    ctx->acc, ctx->cg_r, ctx->cg_p, ctx->cg_q, ctx->hx, ctx->hy, ctx->partials, ctx->scal, ctx->flag};
    for (void* p : ptrs) dev_free(ctx, p);
    for (auto& r : ctx->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    if (ctx->cg_exec) cudaGraphExecDestroy(ctx->cg_exec);
    {
        AmpModel& m = ctx->am;
        PointSources& ps = ctx->pts;
        void* pp[] = {ps.idx, ps.xi, ps.out, ps.flux, ps.dflux, ps.sdiff, ps.stot};
        for (void* q : pp) dev_free(ctx, q);
        void* mp[] = {m.pindex, m.mult, m.d_hyper, m.theta, m.ab, m.wn, m.abf, m.dabf, m.gbin, m.work, m.sc, m.xi};
        for (void* q : mp) dev_free(ctx, q);
    }
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    if (ctx->s_in) {
        cudaStreamDestroy(ctx->s_in); cudaStreamDestroy(ctx->s_out);
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(ctx->ev_in[i]); cudaEventDestroy(ctx->ev_comp[i]); cudaEventDestroy(ctx->ev_out[i]); }
    }
    dev_free(ctx, ctx->hx2);
    dev_free(ctx, ctx->hy2);
    delete ctx;
}

static int build_transposed_weights(frs_ctx* ctx) {
    RET(dev_alloc(ctx, &ctx->wtT, (size_t)ctx->nchan * (ctx->ny / 2 + 1) * 2 * ctx->nx * 2));
    CKL(launch_weights_transpose(ctx->stream, ctx->wt, ctx->wtT, ctx->ny, ctx->nx, ctx->nchan));
    ctx->launches++;
    // both tables exist in natural order now: bring each into the order its column pass consumes
    if (conv_cols_uses_dif(ctx->ny)) {
        CKL(launch_weights_permute(ctx->stream, ctx->wt, ctx->ny, 2 * ctx->ntile, ctx->nchan));
        ctx->launches++;
    }
    if (conv_cols_uses_dif(ctx->nx)) {
        CKL(launch_weights_permute(ctx->stream, ctx->wtT, ctx->nx, 2 * (ctx->ny / 2 + 1), ctx->nchan));
        ctx->launches++;
    }
    return FRS_OK;
}

int frs_set_psf_weights(frs_ctx* ctx, const float* w_half) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !w_half || !aligned16(w_half)) return fail(ctx, FRS_EINVAL, "frs_set_psf_weights: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(dev_alloc(ctx, &ctx->wt, (size_t)ctx->nchan * ctx->ntile * 2 * ctx->ny * 2));
    CK(cudaMemsetAsync(ctx->flag, 0, sizeof(int), ctx->stream));
    CKL(launch_weights_layout(ctx->stream, w_half, ctx->wt, ctx->ny, ctx->nx, ctx->nchan, ctx->flag));
    ctx->launches++;
    RET(build_transposed_weights(ctx));
    int neg = 0;
    CK(cudaMemcpyAsync(&neg, ctx->flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (neg) {
        ctx->have_psf = false;
        return fail(ctx, FRS_ENOTPSD, neg == 2 ? "PSF weights are not Hermitian on the self-conjugate columns kx = 0, nx (W[-k] != W[k])"
                                               : "PSF weights contain negative or NaN entries");
    }
    ctx->have_psf = true;
    ctx->have_kern = false; ctx->lik_mode = 0;    // a kernel fitted to the previous PSF no longer applies
    return FRS_OK;
}

static int set_psf_impl(frs_ctx* ctx, const float* psf, bool covariance);
int frs_set_psf(frs_ctx* ctx, const float* psf) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !psf || !aligned16(psf)) return fail(ctx, FRS_EINVAL, "frs_set_psf: bad argument");
    CK(cudaSetDevice(ctx->device));
    return set_psf_impl(ctx, psf, true);
}

// every point-source pixel inside [0, ly) x [0, lx)?  (a point outside the field of view would have its flux masked to zero
// while the bookkeeping of the latent-space passes kept the unmasked values)
static bool points_inside(const frs_ctx* ctx, int ly, int lx) {
    for (size_t i = 0; i + 1 < ctx->pts_yx.size(); i += 2)
        if (ctx->pts_yx[i] >= ly || ctx->pts_yx[i + 1] >= lx) return false;
    return true;
}

int frs_set_field_of_view(frs_ctx* ctx, int ny_img, int nx_img) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || ny_img < 1 || nx_img < 1 || ny_img > ctx->ny || nx_img > ctx->nx)
        return fail(ctx, FRS_EINVAL, "frs_set_field_of_view: bad argument");
    if (!points_inside(ctx, ny_img, nx_img))
        return fail(ctx, FRS_EINVAL, "frs_set_field_of_view: a point source lies outside the new field of view (frs_set_point_sources first)");
    const bool whole = ny_img == ctx->ny && nx_img == ctx->nx;
    ctx->fov_y = whole ? 0 : ny_img;
    ctx->fov_x = whole ? 0 : nx_img;
    ctx->have_s = ctx->s_ok = ctx->sT_ok = false;
    ctx->am.have_xi = false;
    return FRS_OK;
}

int frs_set_psf_embedded(frs_ctx* ctx, const float* psf_img, int ny_img, int nx_img) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !psf_img || !aligned16(psf_img) || ny_img < 1 || nx_img < 1 || ny_img > ctx->ny || nx_img > ctx->nx)
        return fail(ctx, FRS_EINVAL, "frs_set_psf_embedded: bad argument");
    if (!points_inside(ctx, ny_img, nx_img))
        return fail(ctx, FRS_EINVAL, "frs_set_psf_embedded: a point source lies outside the new field of view (frs_set_point_sources first)");
    CK(cudaSetDevice(ctx->device));
    float* big = nullptr;
    CK(cudaMalloc(reinterpret_cast<void**>(&big), (size_t)ctx->nchan * 4 * ctx->npix * sizeof(float)));
    int rc = FRS_OK;
    const int e = launch_embed_psf(ctx->stream, psf_img, big, ny_img, nx_img, ctx->ny, ctx->nx, ctx->nchan);
    if (e) rc = cuda_fail(ctx, (cudaError_t)e, "launch_embed_psf");
    ctx->launches++;
    // the truncated PSF is real and even but need not be a covariance on the larger grid: its spectrum keeps its sign
    if (rc == FRS_OK) rc = set_psf_impl(ctx, big, false);
    cudaStreamSynchronize(ctx->stream);
    cudaFree(big);
    if (rc != FRS_OK) return rc;
    return frs_set_field_of_view(ctx, ny_img, nx_img);
}

static int set_psf_impl(frs_ctx* ctx, const float* psf, bool covariance) {
    const int my = 2 * ctx->ny, mx = 2 * ctx->nx;
    RET(dev_alloc(ctx, &ctx->wt, (size_t)ctx->nchan * ctx->ntile * 2 * ctx->ny * 2));
    // row pass over all 2 ny rows of length 2 nx (no padding), then one DIF step + ny-point column FFTs
    float2* tmp = nullptr;
    float* stats = nullptr;
    const size_t tstride = spec_batch_stride(my, ctx->nx, kPairBins);
    CK(cudaMalloc(reinterpret_cast<void**>(&tmp), (size_t)ctx->nchan * tstride * sizeof(float2)));
    int rc = FRS_OK;
    std::vector<float> hs;
    int gx = 0;
    auto body = [&]() -> int {
        RowsFwdArgs a{};
        a.in = psf; a.mul = nullptr; a.out = tmp; a.ny = my;
        a.in_bstride = (size_t)my * mx; a.mul_bstride = 0;
        a.scale = 0.5f; a.tw = ctx->tw[ctx->nx]; a.twist = ctx->twist[ctx->nx];
        CKL(launch_rows_fwd(ctx->stream, ctx->nx, false, a, ctx->nchan));
        PsfColsArgs c{};
        c.t = nullptr; c.ntile = ctx->ntile;
        CKL(launch_psf_cols(ctx->stream, ctx->ny, c, ctx->nchan, &gx));   // grid size only
        CK(cudaMalloc(reinterpret_cast<void**>(&stats), (size_t)ctx->nchan * gx * 3 * sizeof(float)));
        c.t = tmp; c.wt = ctx->wt; c.stats = stats; c.scale = 1.0f / ((float)my * (float)mx);
        c.floor = covariance ? 0.f : -3.0e38f;
        c.ncols = ctx->nx + 1; c.w_bstride = (size_t)ctx->ntile * 2 * ctx->ny * 2;
        c.tw = ctx->tw[ctx->ny]; c.twist = ctx->twist[ctx->ny];
        CKL(launch_psf_cols(ctx->stream, ctx->ny, c, ctx->nchan, nullptr));
        ctx->launches += 2;
        RET(build_transposed_weights(ctx));
        hs.resize((size_t)ctx->nchan * gx * 3);
        CK(cudaMemcpyAsync(hs.data(), stats, hs.size() * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
        return FRS_OK;
    };
    rc = body();
    cudaFree(tmp);
    if (stats) cudaFree(stats);
    if (rc != FRS_OK) return rc;
    float max_im = 0.f, min_re = 0.f, max_re = 0.f;
    for (size_t i = 0; i < hs.size(); i += 3) {
        max_im = fmaxf(max_im, hs[i]); min_re = fminf(min_re, hs[i + 1]); max_re = fmaxf(max_re, hs[i + 2]);
    }
    if (!(max_im <= 1e-5f * max_re) || (covariance && !(min_re >= -1e-5f * max_re))) {
        ctx->have_psf = false;
        snprintf(ctx->err, sizeof(ctx->err), "PSF spectrum not real/non-negative: max|Im|=%g min Re=%g max Re=%g", max_im, min_re, max_re);
        return FRS_ENOTPSD;
    }
    ctx->have_psf = true;
    ctx->have_kern = false; ctx->lik_mode = 0;    // a kernel fitted to the previous PSF no longer applies (frs.h, frs_set_noise_kernel)
    return FRS_OK;
}

int frs_set_dirty(frs_ctx* ctx, const float* j) {
    if (!ctx || !j || !aligned16(j)) return fail(ctx, FRS_EINVAL, "frs_set_dirty: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(dev_alloc(ctx, &ctx->dirty, (size_t)ctx->nchan * ctx->npix));
    RET(dev_alloc(ctx, &ctx->dirtyT, (size_t)ctx->nchan * ctx->npix));
    CK(cudaMemcpyAsync(ctx->dirty, j, (size_t)ctx->nchan * ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    RET(transpose(ctx, ctx->dirty, ctx->dirtyT, ctx->ny, ctx->nx, ctx->nchan));
    ctx->have_dirty = true;
    return FRS_OK;
}

int frs_set_amplitude(frs_ctx* ctx, int nfield, const float* amp, const float* mu_host) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !amp || !mu_host || !aligned16(amp) || nfield < 1 || nfield > 2)
        return fail(ctx, FRS_EINVAL, "frs_set_amplitude: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(dev_alloc(ctx, &ctx->amp, 2 * ctx->npix));
    CK(cudaMemcpyAsync(ctx->amp, amp, (size_t)nfield * ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    float mu[2] = {mu_host[0], nfield == 2 ? mu_host[1] : 0.f};
    CK(cudaMemcpyAsync(ctx->d_mu, mu, sizeof(mu), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->nfield = nfield;
    ctx->have_amp = true;
    ctx->have_amp_model = false;          // a fixed amplitude array replaces the learned spectrum
    ctx->have_s = ctx->s_ok = ctx->sT_ok = false;
    return FRS_OK;
}

int frs_set_channel_lognu(frs_ctx* ctx, const float* lognu_host) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !lognu_host) return fail(ctx, FRS_EINVAL, "frs_set_channel_lognu: bad argument");
    CK(cudaSetDevice(ctx->device));
    CK(cudaMemcpyAsync(ctx->d_lognu, lognu_host, ctx->nchan * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->have_s = ctx->s_ok = ctx->sT_ok = false;
    return FRS_OK;
}

int frs_set_sky(frs_ctx* ctx, const float* sky) {
    // no epoch bump: what a new sky can change in the launch sequence of a CG iteration -- the orientation that is valid
    // (sT_ok) and whether point fluxes are in it (pts.in_sky) -- is part of the graph key itself, so a composed model
    // that calls frs_sky_energy_grad every step keeps its captured iteration
    if (!ctx || !sky || !aligned16(sky)) return fail(ctx, FRS_EINVAL, "frs_set_sky: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(ensure_scratch(ctx));
    CK(cudaMemcpyAsync(ctx->s, sky, (size_t)ctx->nchan * ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    if (ctx->fov_y) {
        CKL(launch_mask_outside(ctx->stream, ctx->s, ctx->ny, ctx->nx, ctx->fov_y, ctx->fov_x, ctx->nchan));
        ctx->launches++;
    }
    ctx->have_s = ctx->s_ok = true;
    ctx->sT_ok = false;
    ctx->pts.in_sky = false;              // a sky supplied by the caller has no point-source bookkeeping
    return FRS_OK;
}

int frs_sky_forward(frs_ctx* ctx, const float* xi, float* sky) {
    if (!ctx || !xi || !aligned16(xi) || (sky && !aligned16(sky))) return fail(ctx, FRS_EINVAL, "frs_sky_forward: bad argument");
    if (!ctx->have_amp) return fail(ctx, FRS_ESTATE, "amplitude spectrum not set (frs_set_amplitude)");
    CK(cudaSetDevice(ctx->device));
    RET(ensure_scratch(ctx));
    RET(sky_forward_impl(ctx, xi));
    if (sky) {
        RET(need_s_natural(ctx));
        CK(cudaMemcpyAsync(sky, ctx->s, (size_t)ctx->nchan * ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return FRS_OK;
}

int frs_psf_apply(frs_ctx* ctx, const float* x, float* y) {
    if (!ctx || !x || !y || !aligned16(x) || !aligned16(y)) return fail(ctx, FRS_EINVAL, "frs_psf_apply: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, false, false));
    const Orient o = orient(ctx, false);
    RET(conv_rows_fwd(ctx, o, x, nullptr));
    RET(conv_cols(ctx, o));
    RET(conv_rows_inv(ctx, o, y, kPlain, nullptr, nullptr, nullptr));
    return FRS_OK;
}

int frs_sky_metric_apply(frs_ctx* ctx, const float* x, float* y) {
    if (!ctx || !x || !y || !aligned16(x) || !aligned16(y)) return fail(ctx, FRS_EINVAL, "frs_sky_metric_apply: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, false));
    const Orient o = orient(ctx, false);
    RET(need_s_natural(ctx));
    RET(conv_rows_fwd(ctx, o, x, ctx->s));
    RET(conv_cols(ctx, o));
    RET(conv_rows_inv(ctx, o, y, kMulS, ctx->s, nullptr, nullptr));
    return FRS_OK;
}

static int energy_grad_impl(frs_ctx* ctx, const float* xi, int with_prior, double* d_energy, double* h_energy, float* grad);

int frs_energy_grad(frs_ctx* ctx, const float* xi, int with_prior, double* d_energy, double* h_energy, float* grad) {
    if (!ctx || !xi || !grad || !aligned16(xi) || !aligned16(grad)) return fail(ctx, FRS_EINVAL, "frs_energy_grad: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, false, true));
    if (!ctx->have_dirty) return fail(ctx, FRS_ESTATE, "dirty image not set (frs_set_dirty)");
    return energy_grad_impl(ctx, xi, with_prior, d_energy, h_energy, grad);
}

// the energy is left in ctx->scal[11] (device)
static int energy_grad_impl(frs_ctx* ctx, const float* xi, int with_prior, double* d_energy, double* h_energy, float* grad) {
    RET(sky_forward_impl(ctx, xi));
    const Orient o = orient(ctx, true);                       // sky-space arrays transposed on this path
    if (ctx->lik_mode == 1) {
        // E = 1/2 r^T N'^-1 r, r = j - C s;  grad = -J^T C N'^-1 r (+ xi)        (Eq. 9, R14)
        RET(ensure_scratch9(ctx));
        RET(conv_rows_fwd(ctx, o, ctx->sT, nullptr));
        RET(conv_cols(ctx, o));
        RET(conv_rows_inv(ctx, o, ctx->img2, kResid, nullptr, ctx->dirtyT, nullptr));     // r
        RET(ninv_transposed(ctx, ctx->img2, ctx->img));                                    // u = N'^-1 r
        RET(dot(ctx, ctx->img2, ctx->img, (size_t)ctx->nchan * ctx->npix, ctx->scal + 8));
        if (with_prior) RET(dot(ctx, xi, xi, (size_t)ctx->nfield * ctx->npix, ctx->scal + 10));
        energy9_final_kernel<<<1, 1, 0, ctx->stream>>>(ctx->scal + 8, ctx->scal + 10, with_prior, ctx->scal + 11);
        ctx->launches++;
        RET(conv_rows_fwd(ctx, o, ctx->img, nullptr));
        RET(conv_cols(ctx, o));
        const bool simple = ctx->nchan == 1 && ctx->nfield == 1;
        const bool fused = simple && fused_inv_hart_ok(ctx, o);
        if (fused) {
            RET(conv_rows_inv_hart(ctx, o, kMulS, ctx->sT, nullptr, -1.0f, nullptr));
            RET(hartley_cols(ctx, ctx->nx, ctx->ny, grad, ctx->plain_latent ? nullptr : ctx->amp,
                             (with_prior && !ctx->plain_latent) ? xi : nullptr, nullptr, ctx->nfield));
        } else {
        RET(conv_rows_inv(ctx, o, simple ? ctx->acc : ctx->img, kMulS, ctx->sT, nullptr, nullptr));   // s . C u
        if (simple) RET(points_post(ctx, ctx->acc, -1.0, ctx->scal + 11));
        if (!simple) {
            vjp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->img, ctx->d_lognu, ctx->acc, ctx->npix,
                                                                                   ctx->nfield, ctx->nchan);
            ctx->launches++;
        }
        RET(hartley_t(ctx, ctx->acc, ctx->nx, ctx->ny, nullptr, grad, ctx->plain_latent ? nullptr : ctx->amp,
                      (with_prior && !ctx->plain_latent) ? xi : nullptr, nullptr, ctx->nfield, nullptr, -1.0f));
        }
        CK(cudaGetLastError());
        if (d_energy) CK(cudaMemcpyAsync(d_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        if (h_energy) {
            CK(cudaMemcpyAsync(h_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
        }
        return FRS_OK;
    }
    RET(conv_rows_fwd(ctx, o, ctx->sT, nullptr));
    RET(conv_cols(ctx, o));
    int gx = 0;
    const bool fused0 = fused_inv_hart_ok(ctx, o);
    if (fused0) RET(conv_rows_inv_hart(ctx, o, kEnergy, ctx->sT, ctx->dirtyT, 1.0f, &gx));   // s (C s - j) goes straight into Th
    else
    RET(conv_rows_inv(ctx, o, ctx->img, kEnergy, ctx->sT, ctx->dirtyT, &gx));   // img_c = s_c (C s_c - j_c), partial sums
    const int np = gx;      // one (sum s.c, sum j.s) pair per persistent CTA
    reduce_final_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->partials, np, 2, 0, ctx->scal + 8);
    reduce_final_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->partials, np, 2, 1, ctx->scal + 9);
    ctx->launches += 2;
    if (with_prior) RET(dot(ctx, xi, xi, (size_t)ctx->nfield * ctx->npix, ctx->scal + 10));
    energy_final_kernel<<<1, 1, 0, ctx->stream>>>(ctx->scal + 8, ctx->scal + 9, ctx->scal + 10, with_prior, ctx->scal + 11);
    ctx->launches++;
    if (fused0) {
        RET(hartley_cols(ctx, ctx->nx, ctx->ny, grad, ctx->plain_latent ? nullptr : ctx->amp,
                         (with_prior && !ctx->plain_latent) ? xi : nullptr, nullptr, ctx->nfield));
        CK(cudaGetLastError());
        if (d_energy) CK(cudaMemcpyAsync(d_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        if (h_energy) {
            CK(cudaMemcpyAsync(h_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
        }
        return FRS_OK;
    }
    const float* accp = ctx->img;
    if (ctx->nchan == 1 && ctx->nfield == 1) RET(points_post(ctx, ctx->img, 1.0, ctx->scal + 11));
    if (!(ctx->nchan == 1 && ctx->nfield == 1)) {
        vjp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->img, ctx->d_lognu, ctx->acc, ctx->npix,
                                                                               ctx->nfield, ctx->nchan);
        ctx->launches++;
        accp = ctx->acc;
    }
    RET(hartley_t(ctx, accp, ctx->nx, ctx->ny, nullptr, grad, ctx->plain_latent ? nullptr : ctx->amp,
                  (with_prior && !ctx->plain_latent) ? xi : nullptr, nullptr, ctx->nfield));
    CK(cudaGetLastError());
    if (d_energy) CK(cudaMemcpyAsync(d_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    if (h_energy) {
        CK(cudaMemcpyAsync(h_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
    }
    return FRS_OK;
}

int frs_metric_apply(frs_ctx* ctx, const float* v, int with_prior, float* out) {
    if (!ctx || !v || !out || !aligned16(v) || !aligned16(out) || v == out) return fail(ctx, FRS_EINVAL, "frs_metric_apply: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    return metric_apply_impl(ctx, v, with_prior, out);
}

int frs_cg_read_state(frs_ctx* ctx, float* r, float* p, float* q, double* scal_host) {
    if (!ctx) return FRS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    if (!ctx->have_amp) return fail(ctx, FRS_ESTATE, "amplitude spectrum not set");
    RET(cg_alloc(ctx));
    const size_t bytes = (size_t)ctx->nfield * ctx->npix * sizeof(float);
    if (r) CK(cudaMemcpyAsync(r, ctx->cg_r, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (p) CK(cudaMemcpyAsync(p, ctx->cg_p, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (q) CK(cudaMemcpyAsync(q, ctx->cg_q, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (scal_host) CK(cudaMemcpyAsync(scal_host, ctx->scal, kNScal * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return FRS_OK;
}

int frs_cg_load(frs_ctx* ctx, const float* r, const float* p, double rr_host) {
    if (!ctx || !r || !p) return fail(ctx, FRS_EINVAL, "frs_cg_load: bad argument");
    CK(cudaSetDevice(ctx->device));
    if (!ctx->have_amp) return fail(ctx, FRS_ESTATE, "amplitude spectrum not set");
    RET(cg_alloc(ctx));
    const size_t bytes = (size_t)ctx->nfield * ctx->npix * sizeof(float);
    CK(cudaMemcpyAsync(ctx->cg_r, r, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->cg_p, p, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    double sc[kNScal] = {0};
    sc[kRR] = rr_host;
    CK(cudaMemcpyAsync(ctx->scal, sc, sizeof(sc), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return FRS_OK;
}

int frs_cg_step(frs_ctx* ctx, float* x, int with_prior) {
    if (!ctx || !x || !aligned16(x)) return fail(ctx, FRS_EINVAL, "frs_cg_step: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    RET(cg_alloc(ctx));
    return cg_iter(ctx, x, with_prior, nullptr, 0);
}

int frs_cg_step_begin(frs_ctx* ctx, float** d_q) {
    if (!ctx || !d_q) return fail(ctx, FRS_EINVAL, "frs_cg_step_begin: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    RET(cg_alloc(ctx));
    RET(metric_apply_impl(ctx, ctx->cg_p, 0, ctx->cg_q));
    *d_q = ctx->cg_q;
    return FRS_OK;
}

int frs_cg_step_end(frs_ctx* ctx, float* x, int with_prior) {
    if (!ctx || !x || !aligned16(x)) return fail(ctx, FRS_EINVAL, "frs_cg_step_end: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    RET(cg_alloc(ctx));
    const size_t n = (size_t)ctx->nfield * ctx->npix;
    if (with_prior) {
        add_inplace_kernel<<<(unsigned)((n / 4 + kEwThreads - 1) / kEwThreads + 1), kEwThreads, 0, ctx->stream>>>(ctx->cg_q, ctx->cg_p, n);
        ctx->launches++;
    }
    return cg_iter_finish(ctx, x, nullptr, 0);
}

static int cg_solve_impl(frs_ctx* ctx, const float* b, float* x, int max_iter, float rtol, int with_prior, int* h_iters,
                         double* h_resnorm, double* d_res_history);

int frs_set_fused_passes(frs_ctx* ctx, int on) {
    if (!ctx) return FRS_EINVAL;
    ctx->fuse_inv_hart = on ? 1 : 0;
    ctx->cfg_epoch++;
    return FRS_OK;
}

int frs_set_cuda_graphs(frs_ctx* ctx, int on) {
    if (!ctx) return FRS_EINVAL;
    ctx->use_graphs = on ? 1 : 0;
    return FRS_OK;
}

int frs_cg_solve(frs_ctx* ctx, const float* b, float* x, int max_iter, float rtol, int with_prior, int* h_iters,
                 double* h_resnorm, double* d_res_history) {
    if (!ctx || !b || !x || !aligned16(b) || !aligned16(x) || max_iter < 0 || rtol < 0.f || b == x)
        return fail(ctx, FRS_EINVAL, "frs_cg_solve: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    return cg_solve_impl(ctx, b, x, max_iter, rtol, with_prior, h_iters, h_resnorm, d_res_history);
}

static int cg_solve_impl(frs_ctx* ctx, const float* b, float* x, int max_iter, float rtol, int with_prior, int* h_iters,
                         double* h_resnorm, double* d_res_history) {
    RET(cg_alloc(ctx));
    const size_t n = (size_t)ctx->nfield * ctx->npix;
    const int nb = red_blocks(n);
    CK(cudaMemsetAsync(ctx->scal, 0, kNScal * sizeof(double), ctx->stream));
    CK(cudaMemsetAsync(ctx->scal + kIters, 0, sizeof(double), ctx->stream));
    const double rtol2 = (double)rtol * (double)rtol;
    if (rtol > 0.f) RET(dot(ctx, b, b, n, ctx->scal + kBB));
    // r0 = b - M x0 ; p0 = r0
    RET(metric_apply_impl(ctx, x, with_prior, ctx->cg_q));
    cg_init_kernel<<<nb, kRedThreads, 0, ctx->stream>>>(b, ctx->cg_q, ctx->cg_r, ctx->cg_p, n, ctx->partials);
    reduce_final_kernel<<<1, kRedThreads, 0, ctx->stream>>>(ctx->partials, nb, 1, 0, ctx->scal + kRRNew);
    cg_shift_kernel<<<1, 1, 0, ctx->stream>>>(ctx->scal, d_res_history, 0, rtol2);
    ctx->launches += 3;
    // The stopping test lives on the device; with rtol > 0 the host looks at the flag every 8 iterations only to stop
    // enqueueing (the iterations enqueued past the stopping point leave x, r, p untouched).
    double sc[16];
    // Iteration 0 runs eagerly (it triggers every lazy allocation, tensor map and shared-memory opt-in); the following
    // iterations replay ONE captured iteration as a CUDA graph: at configs 1-2 an iteration is 13 launches of a few
    // microseconds each and the host cannot enqueue them as fast as the device runs them.
    int it = 0;
    if (it < max_iter) {
        RET(cg_iter(ctx, x, with_prior, d_res_history, -1, rtol2));
        ++it;
    }
    const bool graphs = ctx->use_graphs && !ctx->profiling && max_iter - it >= 2;
    if (graphs) {
        // pts_in_sky: whether the cached sky carries point fluxes decides between the fused and the patched launch
        // sequence (points_pre / points_post, fused_inv_hart_ok), and frs_sky_forward / frs_energy_grad flip it
        // without touching the epoch
        const frs_ctx::CgGraphKey key = {x, with_prior, ctx->nfield, ctx->lik_mode, d_res_history, rtol2, ctx->sT_ok,
                                         ctx->pts.n > 0 && ctx->pts.in_sky, ctx->cfg_epoch};
        const frs_ctx::CgGraphKey& k0 = ctx->cg_key;
        const bool same = ctx->cg_exec && k0.x == key.x && k0.with_prior == key.with_prior && k0.nfield == key.nfield &&
                          k0.lik_mode == key.lik_mode && k0.hist == key.hist && k0.rtol2 == key.rtol2 && k0.sT_ok == key.sT_ok &&
                          k0.pts_in_sky == key.pts_in_sky && k0.epoch == key.epoch;
        if (!same) {
            if (ctx->cg_exec) { cudaGraphExecDestroy(ctx->cg_exec); ctx->cg_exec = nullptr; }
            cudaGraph_t g = nullptr;
            const long long l0 = ctx->launches;
            if (!ctx->cap_stream) CK(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
            cudaStream_t user = ctx->stream;
            CK(cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
            ctx->stream = ctx->cap_stream;
            const int rc = cg_iter(ctx, x, with_prior, d_res_history, -1, rtol2);
            ctx->stream = user;
            const cudaError_t ce = cudaStreamEndCapture(ctx->cap_stream, &g);
            ctx->cg_graph_launches = ctx->launches - l0;
            ctx->launches = l0;                     // nothing ran during the capture
            if (rc == FRS_OK && ce == cudaSuccess && g && cudaGraphInstantiate(&ctx->cg_exec, g, 0) == cudaSuccess) {
                ctx->cg_key = key;
            } else {
                ctx->cg_exec = nullptr;
                cudaGetLastError();                 // capture refused: fall back to eager launches below
            }
            if (g) cudaGraphDestroy(g);
        }
    }
    for (; it < max_iter; ++it) {
        if (rtol > 0.f && (it & 7) == 7) {
            CK(cudaMemcpyAsync(sc, ctx->scal, kNScal * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
            if (sc[kDone] != 0.0) break;
        }
        if (graphs && ctx->cg_exec) {
            CK(cudaGraphLaunch(ctx->cg_exec, ctx->stream));
            ctx->launches += ctx->cg_graph_launches;
        } else {
            RET(cg_iter(ctx, x, with_prior, d_res_history, -1, rtol2));
        }
    }
    CK(cudaMemcpyAsync(sc, ctx->scal, 16 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (h_iters) *h_iters = (int)sc[kIters];
    if (h_resnorm) *h_resnorm = sqrt(sc[kRR]);
    if (sc[kBreak] != 0.0) return fail(ctx, FRS_EBREAKDOWN, "CG breakdown: <p, M p> <= 0");
    return FRS_OK;
}

static int latent_scratch(frs_ctx* ctx);
// ---- NEXT-3: learned amplitude spectrum and the joint latent vector (xi, theta)  (Table A.1; reading R17) ----
int frs_amp_model_size(int ny, int nx, int* nb, int* ntheta) {
    if (!pow2_in(ny, 32, 4096) || !pow2_in(nx, 32, 4096) || (!nb && !ntheta)) return FRS_EINVAL;
    const int n = amp_num_bins(ny, nx);
    if (nb) *nb = n;
    if (ntheta) *ntheta = kAmpScalars + 2 * (n - 2);
    return FRS_OK;
}

int frs_set_amplitude_model(frs_ctx* ctx, const float* hyper_host) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !hyper_host) return fail(ctx, FRS_EINVAL, "frs_set_amplitude_model: bad argument");
    if (ctx->nchan != 1) return fail(ctx, FRS_ESTATE, "frs_set_amplitude_model: single-channel contexts only");
    // means of the log-normal parameters must be positive, every standard deviation non-negative
    for (int i = 1; i < kAmpHyper; i += 2)
        if (i != 5 && !(hyper_host[i] > 0.f)) return fail(ctx, FRS_EINVAL, "frs_set_amplitude_model: log-normal mean <= 0");
    for (int i = 2; i < kAmpHyper; i += 2)
        if (!(hyper_host[i] >= 0.f)) return fail(ctx, FRS_EINVAL, "frs_set_amplitude_model: negative standard deviation");
    CK(cudaSetDevice(ctx->device));
    AmpModel& m = ctx->am;
    if (!m.pindex) {
        m.ny = ctx->ny; m.nx = ctx->nx; m.nb = amp_num_bins(ctx->ny, ctx->nx);
        if (m.nb > kAmpMaxBins || m.nb < 4) return fail(ctx, FRS_EINVAL, "frs_set_amplitude_model: unsupported grid");
        RET(dev_alloc(ctx, &m.pindex, ctx->npix));
        RET(dev_alloc(ctx, &m.mult, (size_t)m.nb));
        RET(dev_alloc(ctx, &m.d_hyper, (size_t)kAmpHyper));
        RET(dev_alloc(ctx, &m.theta, (size_t)m.ntheta()));
        RET(dev_alloc(ctx, &m.ab, (size_t)m.nb));
        RET(dev_alloc(ctx, &m.wn, (size_t)m.nb));
        RET(dev_alloc(ctx, &m.abf, (size_t)m.nb));
        RET(dev_alloc(ctx, &m.dabf, (size_t)m.nb));
        RET(dev_alloc(ctx, &m.gbin, (size_t)m.nb));
        RET(dev_alloc(ctx, &m.work, (size_t)4 * m.nb));
        RET(dev_alloc(ctx, &m.sc, (size_t)8));
        RET(dev_alloc(ctx, &m.xi, ctx->npix));
        CKL(launch_amp_bins(ctx->stream, m));
        ctx->launches += 2;
    }
    for (int i = 0; i < kAmpHyper; ++i) m.hyper[i] = (double)hyper_host[i];
    CK(cudaMemcpyAsync(m.d_hyper, m.hyper, sizeof(m.hyper), cudaMemcpyHostToDevice, ctx->stream));
    RET(dev_alloc(ctx, &ctx->amp, 2 * ctx->npix));
    const float mu[2] = {hyper_host[0], 0.f};
    CK(cudaMemcpyAsync(ctx->d_mu, mu, sizeof(mu), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->nfield = 1;
    ctx->have_amp_model = true;
    m.have_theta = m.have_xi = false;
    ctx->have_amp = false;
    ctx->have_s = ctx->s_ok = ctx->sT_ok = false;
    return FRS_OK;
}

static int amp_forward_impl(frs_ctx* ctx, const float* theta) {
    AmpModel& m = ctx->am;
    if (theta != m.theta) CK(cudaMemcpyAsync(m.theta, theta, (size_t)m.ntheta() * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    CKL(launch_amp_forward(ctx->stream, m));
    CKL(launch_amp_gather(ctx->stream, m, m.abf, ctx->amp));
    ctx->launches += 2;
    m.have_theta = true;
    ctx->have_amp = true;
    ctx->have_s = ctx->s_ok = ctx->sT_ok = false;        // the cached sky belongs to the previous amplitude
    m.have_xi = false;
    return FRS_OK;
}

int frs_amplitude_forward(frs_ctx* ctx, const float* theta, float* amp_out) {
    if (!ctx || !theta || (amp_out && !aligned16(amp_out))) return fail(ctx, FRS_EINVAL, "frs_amplitude_forward: bad argument");
    if (!ctx->have_amp_model) return fail(ctx, FRS_ESTATE, "amplitude model not set (frs_set_amplitude_model)");
    CK(cudaSetDevice(ctx->device));
    RET(amp_forward_impl(ctx, theta));
    if (amp_out) CK(cudaMemcpyAsync(amp_out, ctx->amp, ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    return FRS_OK;
}

int frs_amplitude_jvp(frs_ctx* ctx, const float* dtheta, float* d_amp) {
    if (!ctx || !dtheta || !d_amp || !aligned16(d_amp)) return fail(ctx, FRS_EINVAL, "frs_amplitude_jvp: bad argument");
    if (!ctx->have_amp_model || !ctx->am.have_theta) return fail(ctx, FRS_ESTATE, "no amplitude position (frs_amplitude_forward)");
    CK(cudaSetDevice(ctx->device));
    CKL(launch_amp_tangent(ctx->stream, ctx->am, dtheta));
    CKL(launch_amp_gather(ctx->stream, ctx->am, ctx->am.dabf, d_amp));
    ctx->launches += 2;
    return FRS_OK;
}

int frs_amplitude_vjp(frs_ctx* ctx, const float* g_amp, float* g_theta) {
    if (!ctx || !g_amp || !g_theta || !aligned16(g_amp)) return fail(ctx, FRS_EINVAL, "frs_amplitude_vjp: bad argument");
    if (!ctx->have_amp_model || !ctx->am.have_theta) return fail(ctx, FRS_ESTATE, "no amplitude position (frs_amplitude_forward)");
    CK(cudaSetDevice(ctx->device));
    CKL(launch_amp_bin_reduce(ctx->stream, ctx->am, g_amp));
    CKL(launch_amp_adjoint(ctx->stream, ctx->am, nullptr, g_theta, nullptr));
    ctx->launches += 2;
    return FRS_OK;
}

int frs_set_point_sources(frs_ctx* ctx, int npts, const int* yx_host, float alpha, float q) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || npts < 0 || npts > kMaxPoints || (npts > 0 && (!yx_host || !(alpha > 0.f) || !(q > 0.f))))
        return fail(ctx, FRS_EINVAL, "frs_set_point_sources: bad argument");
    if (ctx->nchan != 1) return fail(ctx, FRS_ESTATE, "frs_set_point_sources: single-channel contexts only");
    CK(cudaSetDevice(ctx->device));
    std::vector<int> idx((size_t)npts);
    const int ly = ctx->fov_y ? ctx->fov_y : ctx->ny, lx = ctx->fov_y ? ctx->fov_x : ctx->nx;   // the field of view, not the grid
    for (int i = 0; i < npts; ++i) {
        const int y = yx_host[2 * i], x = yx_host[2 * i + 1];
        if (y < 0 || y >= ly || x < 0 || x >= lx) return fail(ctx, FRS_EINVAL, "frs_set_point_sources: pixel outside the field of view");
        idx[i] = x * ctx->ny + y;                       // the latent-space path keeps the sky transposed
        for (int k = 0; k < i; ++k)
            if (idx[k] == idx[i]) return fail(ctx, FRS_EINVAL, "frs_set_point_sources: the same pixel twice");
    }
    PointSources& p = ctx->pts;
    RET(dev_alloc(ctx, &p.idx, (size_t)kMaxPoints));
    RET(dev_alloc(ctx, &p.xi, (size_t)kMaxPoints));
    RET(dev_alloc(ctx, &p.out, (size_t)kMaxPoints));
    RET(dev_alloc(ctx, &p.flux, (size_t)kMaxPoints));
    RET(dev_alloc(ctx, &p.dflux, (size_t)kMaxPoints));
    RET(dev_alloc(ctx, &p.sdiff, (size_t)kMaxPoints));
    RET(dev_alloc(ctx, &p.stot, (size_t)kMaxPoints));
    if (npts) CK(cudaMemcpyAsync(p.idx, idx.data(), (size_t)npts * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemsetAsync(p.xi, 0, (size_t)kMaxPoints * sizeof(float), ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    p.n = npts; p.alpha = alpha; p.q = q; p.in_sky = false;
    ctx->pts_yx.assign(yx_host, yx_host + 2 * (size_t)npts);
    ctx->have_s = ctx->s_ok = ctx->sT_ok = false;
    ctx->am.have_xi = false;
    return FRS_OK;
}

int frs_energy_grad_joint(frs_ctx* ctx, const float* xi, const float* theta, int with_prior, double* h_energy, float* grad_xi,
                          float* grad_theta) {
    if (!ctx || !xi || !theta || !grad_xi || !grad_theta || !aligned16(xi) || !aligned16(grad_xi) || xi == grad_xi)
        return fail(ctx, FRS_EINVAL, "frs_energy_grad_joint: bad argument");
    if (!ctx->have_amp_model) return fail(ctx, FRS_ESTATE, "amplitude model not set (frs_set_amplitude_model)");
    CK(cudaSetDevice(ctx->device));
    RET(amp_forward_impl(ctx, theta));
    RET(check_hot(ctx, false, true));
    if (!ctx->have_dirty) return fail(ctx, FRS_ESTATE, "dirty image not set (frs_set_dirty)");
    RET(latent_scratch(ctx));
    AmpModel& m = ctx->am;
    const int npts = ctx->pts.n, nta = m.ntheta();      // theta = [amplitude part | point latents]
    if (npts) CK(cudaMemcpyAsync(ctx->pts.xi, theta + nta, (size_t)npts * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaMemcpyAsync(m.xi, xi, ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    m.have_xi = true;
    // h = H[s (C s - j)] (mode 0) or -H[s C N'^-1 r] (mode 1): the latent-space passes without their fused . A + xi
    ctx->plain_latent = true;
    ctx->pts_add = (npts && with_prior) ? ctx->pts.xi : nullptr;
    ctx->pts_out = npts ? grad_theta + nta : nullptr;
    const int rc = energy_grad_impl(ctx, xi, with_prior, nullptr, nullptr, ctx->lat1);
    ctx->plain_latent = false;
    ctx->pts_add = nullptr;
    ctx->pts_out = nullptr;
    RET(rc);
    // grad_xi = A . h (+ xi);  G_b = bin sums of xi . h;  grad_theta = (dA/dtheta)^T G (+ theta);  E += 1/2 <theta, theta>
    CKL(launch_joint_epilogue(ctx->stream, m, ctx->lat1, xi, with_prior ? xi : nullptr, grad_xi));
    CKL(launch_amp_adjoint(ctx->stream, m, with_prior ? m.theta : nullptr, grad_theta, with_prior ? ctx->scal + 11 : nullptr));
    ctx->launches += 2;
    if (h_energy) {
        CK(cudaMemcpyAsync(h_energy, ctx->scal + 11, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
    }
    return FRS_OK;
}

int frs_metric_apply_joint(frs_ctx* ctx, const float* dxi, const float* dtheta, int with_prior, float* out_xi, float* out_theta) {
    if (!ctx || !dxi || !dtheta || !out_xi || !out_theta || !aligned16(dxi) || !aligned16(out_xi) || dxi == out_xi)
        return fail(ctx, FRS_EINVAL, "frs_metric_apply_joint: bad argument");
    if (!ctx->have_amp_model || !ctx->am.have_theta || !ctx->am.have_xi)
        return fail(ctx, FRS_ESTATE, "no joint position (frs_energy_grad_joint)");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    RET(latent_scratch(ctx));
    AmpModel& m = ctx->am;
    // u = A . dxi + dA(dtheta) . xi;  h = H[s C s H[u]] (mode 0; mode 1 with N'^-1 in the middle)
    CKL(launch_amp_tangent(ctx->stream, m, dtheta));
    CKL(launch_joint_prologue(ctx->stream, m, dxi, m.xi, ctx->lat1));
    ctx->launches += 2;
    const int npts = ctx->pts.n, nta = m.ntheta();
    ctx->plain_latent = true;
    ctx->pts_dv = npts ? dtheta + nta : nullptr;
    ctx->pts_add = (npts && with_prior) ? dtheta + nta : nullptr;
    ctx->pts_out = npts ? out_theta + nta : nullptr;
    const int rc = metric_apply_impl(ctx, ctx->lat1, with_prior, ctx->lat2);
    ctx->plain_latent = false;
    ctx->pts_dv = ctx->pts_add = nullptr;
    ctx->pts_out = nullptr;
    RET(rc);
    CKL(launch_joint_epilogue(ctx->stream, m, ctx->lat2, m.xi, with_prior ? dxi : nullptr, out_xi));
    CKL(launch_amp_adjoint(ctx->stream, m, with_prior ? dtheta : nullptr, out_theta, nullptr));
    ctx->launches += 2;
    return FRS_OK;
}

// ---- building blocks of composed sky models: several Gaussian processes on patches (reading R20) --------------
// A composed model keeps one context per component (its own grid, amplitude and position) and one for the full field;
// these calls expose the two halves the existing calls fuse: the sky-space derivative of the likelihood and the Jacobian
// of one log-normal field.
int frs_sky_energy_grad(frs_ctx* ctx, const float* sky, double* h_energy, float* grad_sky) {
    if (!ctx || !sky || !grad_sky || !aligned16(sky) || !aligned16(grad_sky) || sky == grad_sky)
        return fail(ctx, FRS_EINVAL, "frs_sky_energy_grad: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(frs_set_sky(ctx, sky));
    RET(check_hot(ctx, true, false));
    if (!ctx->have_dirty) return fail(ctx, FRS_ESTATE, "dirty image not set (frs_set_dirty)");
    const Orient o = orient(ctx, false);
    const size_t n = (size_t)ctx->nchan * ctx->npix;
    const unsigned eg = (unsigned)((n / 4 + kEwThreads - 1) / kEwThreads);
    RET(ensure_scratch9(ctx));
    RET(conv_rows_fwd(ctx, o, ctx->s, nullptr));
    RET(conv_cols(ctx, o));
    RET(conv_rows_inv(ctx, o, ctx->img2, kResid, nullptr, ctx->dirty, nullptr));            // r = j - C s
    if (ctx->lik_mode == 0) {
        // E = 1/2 <s, C s> - <j, s> = -1/2 <s, r> - 1/2 <j, s>;  dE/ds = C s - j = -r
        RET(dot(ctx, ctx->s, ctx->img2, n, ctx->scal + 8));
        RET(dot(ctx, ctx->dirty, ctx->s, n, ctx->scal + 9));
        accumulate_kernel<<<eg, kEwThreads, 0, ctx->stream>>>(grad_sky, ctx->img2, -1.0f, 1, n, nullptr, nullptr);
        ctx->launches++;
    } else {
        // E = 1/2 r^T N'^-1 r;  dE/ds = -C N'^-1 r
        if (!ctx->have_kern) return fail(ctx, FRS_ESTATE, "noise kernel not set (frs_set_noise_kernel)");
        RET(hartley_t(ctx, ctx->img2, ctx->ny, ctx->nx, nullptr, ctx->img3, ctx->kinvT, nullptr, nullptr, ctx->nchan));
        RET(hartley_t(ctx, ctx->img3, ctx->nx, ctx->ny, nullptr, ctx->img, nullptr, nullptr, nullptr, ctx->nchan));   // u
        RET(dot(ctx, ctx->img2, ctx->img, n, ctx->scal + 8));
        RET(conv_rows_fwd(ctx, o, ctx->img, nullptr));
        RET(conv_cols(ctx, o));
        RET(conv_rows_inv(ctx, o, ctx->img3, kPlain, nullptr, nullptr, nullptr));
        accumulate_kernel<<<eg, kEwThreads, 0, ctx->stream>>>(grad_sky, ctx->img3, -1.0f, 1, n, nullptr, nullptr);
        ctx->launches++;
    }
    CK(cudaGetLastError());
    if (h_energy) {
        double sc[2];
        CK(cudaMemcpyAsync(sc, ctx->scal + 8, sizeof(sc), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
        *h_energy = ctx->lik_mode == 0 ? -0.5 * sc[0] - 0.5 * sc[1] : 0.5 * sc[0];
    }
    return FRS_OK;
}

// dsky = s . H[A v] at the cached position (natural orientation)
int frs_latent_jvp(frs_ctx* ctx, const float* v, float* dsky) {
    if (!ctx || !v || !dsky || !aligned16(v) || !aligned16(dsky)) return fail(ctx, FRS_EINVAL, "frs_latent_jvp: bad argument");
    if (ctx->nchan != 1 || ctx->nfield != 1) return fail(ctx, FRS_ESTATE, "frs_latent_jvp: single channel, one field");
    CK(cudaSetDevice(ctx->device));
    if (!ctx->have_amp || !ctx->have_s) return fail(ctx, FRS_ESTATE, "no position (frs_sky_forward)");
    RET(ensure_scratch(ctx));
    RET(need_s_transposed(ctx));
    RET(hartley_t(ctx, v, ctx->ny, ctx->nx, ctx->amp, ctx->lin, nullptr, nullptr, nullptr, 1));      // [nx][ny]
    mul_inplace_kernel<<<(unsigned)((ctx->npix / 4 + kEwThreads - 1) / kEwThreads), kEwThreads, 0, ctx->stream>>>(ctx->lin, ctx->sT, ctx->npix);
    ctx->launches++;
    RET(transpose(ctx, ctx->lin, dsky, ctx->nx, ctx->ny, 1));
    return FRS_OK;
}

// out = A . H[s . w] (+ add) at the cached position; w in the natural orientation
int frs_latent_vjp(frs_ctx* ctx, const float* w_sky, const float* add, float* out) {
    if (!ctx || !w_sky || !out || !aligned16(w_sky) || !aligned16(out) || (add && !aligned16(add)))
        return fail(ctx, FRS_EINVAL, "frs_latent_vjp: bad argument");
    if (ctx->nchan != 1 || ctx->nfield != 1) return fail(ctx, FRS_ESTATE, "frs_latent_vjp: single channel, one field");
    CK(cudaSetDevice(ctx->device));
    if (!ctx->have_amp || !ctx->have_s) return fail(ctx, FRS_ESTATE, "no position (frs_sky_forward)");
    RET(ensure_scratch(ctx));
    RET(need_s_transposed(ctx));
    RET(transpose(ctx, w_sky, ctx->img, ctx->ny, ctx->nx, 1));                                       // [nx][ny]
    RET(hartley_t(ctx, ctx->img, ctx->nx, ctx->ny, ctx->sT, out, ctx->amp, add, nullptr, 1));
    return FRS_OK;
}

// <a, b> over n floats (n a multiple of 4), accumulated in fp64 with the fixed-order reduction of the CG scalars
int frs_dot(frs_ctx* ctx, const float* a, const float* b, long long n, double* h_out) {
    if (!ctx || !a || !b || !h_out || n <= 0 || (n & 3) || !aligned16(a) || !aligned16(b)) return fail(ctx, FRS_EINVAL, "frs_dot: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(ensure_scratch(ctx));
    RET(dot(ctx, a, b, (size_t)n, ctx->scal + 14));
    CK(cudaMemcpyAsync(h_out, ctx->scal + 14, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return FRS_OK;
}

int frs_patch_insert_add(frs_ctx* ctx, const float* patch, int nyp, int nxp, int y0, int x0, float* field) {
    if (!ctx || !patch || !field || nyp < 1 || nxp < 1 || y0 < 0 || x0 < 0 || y0 + nyp > ctx->ny || x0 + nxp > ctx->nx)
        return fail(ctx, FRS_EINVAL, "frs_patch_insert_add: patch outside the field");
    CK(cudaSetDevice(ctx->device));
    CKL(launch_patch_copy(ctx->stream, field, ctx->ny, ctx->nx, const_cast<float*>(patch), nyp, nxp, y0, x0, 1));
    ctx->launches++;
    return FRS_OK;
}
int frs_patch_crop(frs_ctx* ctx, const float* field, int nyp, int nxp, int y0, int x0, float* patch) {
    if (!ctx || !patch || !field || nyp < 1 || nxp < 1 || y0 < 0 || x0 < 0 || y0 + nyp > ctx->ny || x0 + nxp > ctx->nx)
        return fail(ctx, FRS_EINVAL, "frs_patch_crop: patch outside the field");
    CK(cudaSetDevice(ctx->device));
    CKL(launch_patch_copy(ctx->stream, const_cast<float*>(field), ctx->ny, ctx->nx, patch, nyp, nxp, y0, x0, 0));
    ctx->launches++;
    return FRS_OK;
}

// ---- MGVI: posterior samples and the sample-averaged KL (reading R15) ------------------------
static int latent_scratch(frs_ctx* ctx) {
    RET(dev_alloc(ctx, &ctx->lat1, 2 * ctx->npix));
    RET(dev_alloc(ctx, &ctx->lat2, 2 * ctx->npix));
    return FRS_OK;
}

int frs_draw_sample(frs_ctx* ctx, const float* eta_xi, const float* eta_d, int max_iter, float rtol, float* sample, int* h_iters) {
    if (!ctx || !eta_xi || !eta_d || !sample || !aligned16(eta_xi) || !aligned16(eta_d) || !aligned16(sample) || max_iter < 0 ||
        rtol < 0.f || sample == eta_xi)
        return fail(ctx, FRS_EINVAL, "frs_draw_sample: bad argument");
    if (ctx->lik_mode != 1) return fail(ctx, FRS_ESTATE, "frs_draw_sample needs the Eq. 9 likelihood (frs_set_likelihood(ctx, 1))");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, true));
    RET(ensure_scratch9(ctx));
    RET(latent_scratch(ctx));
    const Orient o = orient(ctx, true);
    RET(need_s_transposed(ctx));
    // m = eta_xi + J^T C N'^-1/2 eta_d  (Cov m = M): the sky-space chain runs in the transposed orientation
    RET(transpose(ctx, eta_d, ctx->img2, ctx->ny, ctx->nx, ctx->nchan));
    RET(hartley_t(ctx, ctx->img2, ctx->nx, ctx->ny, nullptr, ctx->img3, ctx->kisqN, nullptr, nullptr, ctx->nchan));
    RET(hartley_t(ctx, ctx->img3, ctx->ny, ctx->nx, nullptr, ctx->img, nullptr, nullptr, nullptr, ctx->nchan));
    RET(conv_rows_fwd(ctx, o, ctx->img, nullptr));
    RET(conv_cols(ctx, o));
    const bool simple = ctx->nchan == 1 && ctx->nfield == 1;
    RET(conv_rows_inv(ctx, o, simple ? ctx->acc : ctx->img, kMulS, ctx->sT, nullptr, nullptr));
    if (simple) {
        // J^T of the metric the CG below inverts is the DIFFUSE Jacobian at the point-source pixels (metric_apply_impl):
        // the source must be formed with the same one, or Cov m != M there
        RET(points_post(ctx, ctx->acc, 1.0, nullptr));
    } else {
        vjp_combine_kernel<<<ew_grid(ctx->npix), kEwThreads, 0, ctx->stream>>>(ctx->img, ctx->d_lognu, ctx->acc, ctx->npix,
                                                                               ctx->nfield, ctx->nchan);
        ctx->launches++;
    }
    RET(hartley_t(ctx, ctx->acc, ctx->nx, ctx->ny, nullptr, ctx->lat1, ctx->amp, eta_xi, nullptr, ctx->nfield));
    // sigma = M^-1 m by CG from 0.  The solve runs in a buffer of the context's own and is copied out: the captured CG
    // iteration is keyed on the solution pointer, and callers hand in a fresh `sample` buffer per draw
    // (SampleShard.draw), which would re-capture the graph on every sample
    const size_t nbytes = (size_t)ctx->nfield * ctx->npix * sizeof(float);
    CK(cudaMemsetAsync(ctx->lat2, 0, nbytes, ctx->stream));
    const int rc = cg_solve_impl(ctx, ctx->lat1, ctx->lat2, max_iter, rtol, 1, h_iters, nullptr, nullptr);
    CK(cudaMemcpyAsync(sample, ctx->lat2, nbytes, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return rc;
}

int frs_kl_energy_grad(frs_ctx* ctx, const float* xi, const float* samples, int nsamples, int mirrored, double* d_energy,
                       double* h_energy, float* grad) {
    if (!ctx || !xi || !samples || !grad || nsamples < 1 || !aligned16(xi) || !aligned16(samples) || !aligned16(grad) || grad == xi)
        return fail(ctx, FRS_EINVAL, "frs_kl_energy_grad: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, false, true));
    if (!ctx->have_dirty) return fail(ctx, FRS_ESTATE, "dirty image not set (frs_set_dirty)");
    RET(latent_scratch(ctx));
    const size_t n = (size_t)ctx->nfield * ctx->npix;
    RET(for_each_position(ctx, xi, samples, nsamples, mirrored, [&](const float* q, float w, bool first) -> int {
        RET(energy_grad_impl(ctx, q, 1, nullptr, nullptr, ctx->lat2));
        accumulate_kernel<<<ew_grid(n), kEwThreads, 0, ctx->stream>>>(grad, ctx->lat2, w, first ? 1 : 0, n, ctx->scal + 13, ctx->scal + 11);
        ctx->launches++;
        return FRS_OK;
    }));
    RET(sky_forward_impl(ctx, xi));                           // leave the position at the mean
    CK(cudaGetLastError());
    if (d_energy) CK(cudaMemcpyAsync(d_energy, ctx->scal + 13, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    if (h_energy) {
        CK(cudaMemcpyAsync(h_energy, ctx->scal + 13, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaStreamSynchronize(ctx->stream));
    }
    return FRS_OK;
}

int frs_kl_metric_apply(frs_ctx* ctx, const float* xi, const float* samples, int nsamples, int mirrored, const float* v, float* out) {
    if (!ctx || !xi || !samples || !v || !out || nsamples < 1 || !aligned16(xi) || !aligned16(samples) || !aligned16(v) ||
        !aligned16(out) || out == v || out == xi)
        return fail(ctx, FRS_EINVAL, "frs_kl_metric_apply: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, false, true));
    RET(latent_scratch(ctx));
    const size_t n = (size_t)ctx->nfield * ctx->npix;
    RET(for_each_position(ctx, xi, samples, nsamples, mirrored, [&](const float* q, float w, bool first) -> int {
        RET(sky_forward_impl(ctx, q));
        RET(metric_apply_impl(ctx, v, 1, ctx->lat2));
        accumulate_kernel<<<ew_grid(n), kEwThreads, 0, ctx->stream>>>(out, ctx->lat2, w, first ? 1 : 0, n, nullptr, nullptr);
        ctx->launches++;
        return FRS_OK;
    }));
    RET(sky_forward_impl(ctx, xi));
    CK(cudaGetLastError());
    return FRS_OK;
}

// ---- major cycle: exact response on uv points (Alg. 1, Eq. 20-22; reading R16) ----------------------
static int response_args(frs_ctx* ctx, const float* uv, const float* wgt, int nvis, const char* who) {
    if (!ctx) return FRS_EINVAL;
    if (!uv || nvis < 1 || (reinterpret_cast<uintptr_t>(uv) & 7u) || (wgt && (reinterpret_cast<uintptr_t>(wgt) & 3u))) return fail(ctx, FRS_EINVAL, who);
    if (ctx->ny > kMaxResponseSide || ctx->nx > kMaxResponseSide)
        return fail(ctx, FRS_EINVAL, "exact response: direct sums are provided for ny, nx <= 1024 (O(nvis npix); larger fields need a gridder)");
    return FRS_OK;
}

int frs_exact_response(frs_ctx* ctx, const float* uv, int nvis, const float* x, float* vis) {
    RET(response_args(ctx, uv, nullptr, nvis, "frs_exact_response: bad argument"));
    if (!x || !vis || (reinterpret_cast<uintptr_t>(vis) & 7u)) return fail(ctx, FRS_EINVAL, "frs_exact_response: bad argument");
    CK(cudaSetDevice(ctx->device));
    CKL(launch_exact_degrid(ctx->stream, uv, nvis, x, ctx->ny, ctx->nx, vis));
    ctx->launches++;
    return FRS_OK;
}

int frs_exact_adjoint(frs_ctx* ctx, const float* uv, const float* wgt, int nvis, const float* vis, float* y) {
    RET(response_args(ctx, uv, wgt, nvis, "frs_exact_adjoint: bad argument"));
    if (!wgt || !vis || !y || (reinterpret_cast<uintptr_t>(vis) & 7u)) return fail(ctx, FRS_EINVAL, "frs_exact_adjoint: bad argument");
    CK(cudaSetDevice(ctx->device));
    CKL(launch_exact_grid(ctx->stream, uv, wgt, vis, nvis, ctx->ny, ctx->nx, nullptr, 1.0f, y));
    ctx->launches++;
    return FRS_OK;
}

int frs_major_cycle_residual(frs_ctx* ctx, const float* uv, const float* wgt, int nvis, const float* dirty_full, const float* sky,
                             float* d_next) {
    RET(response_args(ctx, uv, wgt, nvis, "frs_major_cycle_residual: bad argument"));
    if (!wgt || !dirty_full || !sky || !d_next) return fail(ctx, FRS_EINVAL, "frs_major_cycle_residual: bad argument");
    CK(cudaSetDevice(ctx->device));
    if (ctx->visbuf_n < (size_t)nvis) {
        if (ctx->visbuf) dev_free(ctx, ctx->visbuf);
        ctx->visbuf = nullptr;
        CK(cudaMalloc(reinterpret_cast<void**>(&ctx->visbuf), (size_t)nvis * 2 * sizeof(float)));
        ctx->visbuf_n = (size_t)nvis;
    }
    // d_{i+1} = I^D - R^+ N^-1 R I_i
    CKL(launch_exact_degrid(ctx->stream, uv, nvis, sky, ctx->ny, ctx->nx, ctx->visbuf));
    CKL(launch_exact_grid(ctx->stream, uv, wgt, ctx->visbuf, nvis, ctx->ny, ctx->nx, dirty_full, -1.0f, d_next));
    ctx->launches += 2;
    return FRS_OK;
}

// ---- the paper's literal likelihood: noise kernel of Eq. 15-18 ------------------------------------
static int kernel_arrays(frs_ctx* ctx) {
    const size_t n = (size_t)ctx->nchan * ctx->npix;
    RET(dev_alloc(ctx, &ctx->kern, n));
    RET(dev_alloc(ctx, &ctx->kinvN, n));
    RET(dev_alloc(ctx, &ctx->kinvT, n));
    RET(dev_alloc(ctx, &ctx->kisqN, n));
    return ensure_scratch9(ctx);
}

int frs_set_noise_kernel(frs_ctx* ctx, float eps) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !(eps > 0.f)) return fail(ctx, FRS_EINVAL, "frs_set_noise_kernel: eps must be > 0");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, false, false));
    RET(kernel_arrays(ctx));
    const size_t n = (size_t)ctx->nchan * ctx->npix;
    // t = C I_delta with the point source in the centre of the field (Eq. 17), one per channel
    CK(cudaMemsetAsync(ctx->img2, 0, n * sizeof(float), ctx->stream));
    set_delta_kernel<<<ctx->nchan, 1, 0, ctx->stream>>>(ctx->img2, ctx->npix, (size_t)(ctx->ny / 2) * ctx->nx + ctx->nx / 2);
    ctx->launches++;
    const Orient o = orient(ctx, false);
    RET(conv_rows_fwd(ctx, o, ctx->img2, nullptr));
    RET(conv_cols(ctx, o));
    RET(conv_rows_inv(ctx, o, ctx->img, kPlain, nullptr, nullptr, nullptr));
    RET(hartley_t(ctx, ctx->img, ctx->ny, ctx->nx, nullptr, ctx->img3, nullptr, nullptr, nullptr, ctx->nchan));   // [nx][ny]
    dim3 grid((unsigned)((ctx->npix + 255) / 256), ctx->nchan);
    noise_kernel_finish_kernel<<<grid, 256, 0, ctx->stream>>>(ctx->img3, eps, ctx->kern, ctx->kinvN, ctx->kinvT, ctx->kisqN, ctx->ny, ctx->nx);
    ctx->launches++;
    CK(cudaGetLastError());
    ctx->have_kern = true;
    return FRS_OK;
}

int frs_set_noise_kernel_array(frs_ctx* ctx, const float* kern) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || !kern || !aligned16(kern)) return fail(ctx, FRS_EINVAL, "frs_set_noise_kernel_array: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(ensure_scratch(ctx));
    RET(kernel_arrays(ctx));
    const size_t n = (size_t)ctx->nchan * ctx->npix;
    CK(cudaMemcpyAsync(ctx->kern, kern, n * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaMemsetAsync(ctx->flag, 0, sizeof(int), ctx->stream));
    dim3 grid((unsigned)((ctx->npix + 255) / 256), ctx->nchan);
    noise_kernel_from_array_kernel<<<grid, 256, 0, ctx->stream>>>(ctx->kern, ctx->kinvN, ctx->kinvT, ctx->kisqN, ctx->ny, ctx->nx, ctx->flag);
    ctx->launches++;
    int bad = 0;
    CK(cudaMemcpyAsync(&bad, ctx->flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (bad) { ctx->have_kern = false; return fail(ctx, FRS_ENOTPSD, "noise kernel must be > 0 and even (K[-k] = K[k])"); }
    ctx->have_kern = true;
    return FRS_OK;
}

int frs_get_noise_kernel(frs_ctx* ctx, float* kern) {
    if (!ctx || !kern || !aligned16(kern)) return fail(ctx, FRS_EINVAL, "frs_get_noise_kernel: bad argument");
    if (!ctx->have_kern) return fail(ctx, FRS_ESTATE, "noise kernel not set (frs_set_noise_kernel)");
    CK(cudaSetDevice(ctx->device));
    CK(cudaMemcpyAsync(kern, ctx->kern, (size_t)ctx->nchan * ctx->npix * sizeof(float), cudaMemcpyDeviceToDevice, ctx->stream));
    return FRS_OK;
}

int frs_ninv_apply(frs_ctx* ctx, const float* x, float* y) {
    if (!ctx || !x || !y || !aligned16(x) || !aligned16(y)) return fail(ctx, FRS_EINVAL, "frs_ninv_apply: bad argument");
    if (!ctx->have_kern) return fail(ctx, FRS_ESTATE, "noise kernel not set (frs_set_noise_kernel)");
    CK(cudaSetDevice(ctx->device));
    RET(ensure_scratch(ctx));
    RET(hartley_t(ctx, x, ctx->ny, ctx->nx, nullptr, ctx->img3, ctx->kinvT, nullptr, nullptr, ctx->nchan));   // [nx][ny]
    RET(hartley_t(ctx, ctx->img3, ctx->nx, ctx->ny, nullptr, y, nullptr, nullptr, nullptr, ctx->nchan));
    return FRS_OK;
}

int frs_set_likelihood(frs_ctx* ctx, int mode) {
    if (ctx) ctx->cfg_epoch++;
    if (!ctx || (mode != 0 && mode != 1)) return fail(ctx, FRS_EINVAL, "frs_set_likelihood: mode must be 0 or 1");
    if (mode == 1 && !ctx->have_kern) return fail(ctx, FRS_ESTATE, "noise kernel not set (frs_set_noise_kernel)");
    ctx->lik_mode = mode;
    return FRS_OK;
}

static int host_apply(frs_ctx* ctx, const float* xh, float* yh, bool with_s) {
    if (!ctx || !xh || !yh) return fail(ctx, FRS_EINVAL, "host apply: bad argument");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, with_s, false));
    const size_t n = (size_t)ctx->nchan * ctx->npix;
    RET(dev_alloc(ctx, &ctx->hx, n));
    RET(dev_alloc(ctx, &ctx->hy, n));
    CK(cudaMemcpyAsync(ctx->hx, xh, n * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    const Orient o = orient(ctx, false);
    if (with_s) RET(need_s_natural(ctx));
    RET(conv_rows_fwd(ctx, o, ctx->hx, with_s ? ctx->s : nullptr));
    RET(conv_cols(ctx, o));
    RET(conv_rows_inv(ctx, o, ctx->hy, with_s ? kMulS : kPlain, ctx->s, nullptr, nullptr));
    CK(cudaMemcpyAsync(yh, ctx->hy, n * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return FRS_OK;
}
int frs_sky_metric_apply_host(frs_ctx* ctx, const float* x_host, float* y_host) { return host_apply(ctx, x_host, y_host, true); }

// n independent applies with the copies of neighbouring items overlapping the kernels: host -> device of item k + 1 and
// device -> host of item k - 1 run on two copy streams of the ctx's own while item k computes (two device buffers each way)
int frs_sky_metric_apply_host_batch(frs_ctx* ctx, int n, const float* const* x_hosts, float* const* y_hosts) {
    if (!ctx || n < 0 || (n > 0 && (!x_hosts || !y_hosts))) return fail(ctx, FRS_EINVAL, "frs_sky_metric_apply_host_batch: bad argument");
    for (int k = 0; k < n; ++k)
        if (!x_hosts[k] || !y_hosts[k]) return fail(ctx, FRS_EINVAL, "frs_sky_metric_apply_host_batch: null buffer");
    CK(cudaSetDevice(ctx->device));
    RET(check_hot(ctx, true, false));
    const size_t cnt = (size_t)ctx->nchan * ctx->npix;
    RET(dev_alloc(ctx, &ctx->hx, cnt));
    RET(dev_alloc(ctx, &ctx->hy, cnt));
    RET(dev_alloc(ctx, &ctx->hx2, cnt));
    RET(dev_alloc(ctx, &ctx->hy2, cnt));
    if (!ctx->s_in) {
        CK(cudaStreamCreateWithFlags(&ctx->s_in, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&ctx->s_out, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CK(cudaEventCreateWithFlags(&ctx->ev_in[i], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&ctx->ev_comp[i], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&ctx->ev_out[i], cudaEventDisableTiming));
        }
    }
    RET(need_s_natural(ctx));
    const Orient o = orient(ctx, false);
    float* hx[2] = {ctx->hx, ctx->hx2};
    float* hy[2] = {ctx->hy, ctx->hy2};
    // everything enqueued so far on the ctx's stream (the sky, the spectrum) precedes the first copy
    CK(cudaEventRecord(ctx->ev_comp[0], ctx->stream));
    CK(cudaEventRecord(ctx->ev_comp[1], ctx->stream));
    bool out_used[2] = {false, false};
    for (int k = 0; k < n; ++k) {
        const int b = k & 1;
        CK(cudaStreamWaitEvent(ctx->s_in, ctx->ev_comp[b], 0));               // item k - 2 has read hx[b]
        CK(cudaMemcpyAsync(hx[b], x_hosts[k], cnt * sizeof(float), cudaMemcpyHostToDevice, ctx->s_in));
        CK(cudaEventRecord(ctx->ev_in[b], ctx->s_in));
        CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_in[b], 0));
        if (out_used[b]) CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_out[b], 0));   // item k - 2 has left hy[b]
        RET(conv_rows_fwd(ctx, o, hx[b], ctx->s));
        RET(conv_cols(ctx, o));
        RET(conv_rows_inv(ctx, o, hy[b], kMulS, ctx->s, nullptr, nullptr));
        CK(cudaEventRecord(ctx->ev_comp[b], ctx->stream));
        CK(cudaStreamWaitEvent(ctx->s_out, ctx->ev_comp[b], 0));
        CK(cudaMemcpyAsync(y_hosts[k], hy[b], cnt * sizeof(float), cudaMemcpyDeviceToHost, ctx->s_out));
        CK(cudaEventRecord(ctx->ev_out[b], ctx->s_out));
        out_used[b] = true;
    }
    CK(cudaStreamSynchronize(ctx->s_out));
    CK(cudaStreamSynchronize(ctx->stream));
    return FRS_OK;
}
int frs_psf_apply_host(frs_ctx* ctx, const float* x_host, float* y_host) { return host_apply(ctx, x_host, y_host, false); }

// number of ctx-owned arrays whose guard zones were written to (0 without FRS_GUARD=1); *n_arrays: arrays under guard
int frs_debug_check_guards(frs_ctx* ctx, int* n_arrays) {
    if (!ctx) return -1;
    CK(cudaSetDevice(ctx->device));
    CK(cudaDeviceSynchronize());
    int bad = 0, n = 0;
    std::vector<unsigned char> h;
    for (const auto& g : ctx->guards) {
        if (!g.base) continue;
        ++n;
        const size_t tail = g.padded - g.used + kGuardBytes;
        h.resize(kGuardBytes + tail);
        if (cudaMemcpy(h.data(), g.base, kGuardBytes, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
        if (cudaMemcpy(h.data() + kGuardBytes, g.base + kGuardBytes + g.used, tail, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
        bool ok = true;
        for (unsigned char c : h) ok = ok && c == (unsigned char)kGuardByte;
        if (!ok) ++bad;
    }
    if (n_arrays) *n_arrays = n;
    return bad;
}

int frs_profile_enable(frs_ctx* ctx, int on) {
    if (!ctx) return FRS_EINVAL;
    ctx->profiling = on != 0;
    return FRS_OK;
}

int frs_profile_read(frs_ctx* ctx, double ms[5], long long launches[5]) {
    if (!ctx || !ms || !launches) return FRS_EINVAL;
    CK(cudaSetDevice(ctx->device));
    CK(cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < kNPass; ++i) { ms[i] = 0.0; launches[i] = 0; }
    for (auto& r : ctx->prof) {
        float t = 0.f;
        cudaEventElapsedTime(&t, r.a, r.b);
        ms[r.kind] += t;
        launches[r.kind]++;
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    ctx->prof.clear();
    return FRS_OK;
}

}  // extern "C"
