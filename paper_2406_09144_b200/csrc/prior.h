// prior.h -- learned amplitude spectrum of the diffuse-emission prior (NEXT-3, Table A.1 P:536-550;
// DESIGN.md reading R17).  Launchers of k_prior.cu; every pointer is a device pointer unless it says host.
#pragma once
#include <cuda_runtime.h>

namespace frs {

constexpr int kAmpScalars = 5;      // xi_fluct, xi_slope, xi_flex, xi_asp, xi_zm
constexpr int kAmpHyper = 11;       // offset, zm mean/std, fluct mean/std, slope mean/std, flex mean/std, asp mean/std
constexpr int kAmpMaxBins = 8192;   // one CTA scans the spectrum; 4096^2 has 2897 bins

// radial bins of an ny x nx harmonic grid: number of bins (host arithmetic only)
int amp_num_bins(int ny, int nx);

struct AmpModel {
    int ny = 0, nx = 0, nb = 0;
    unsigned short* pindex = nullptr;   // [ny][nx] bin of every mode (nb <= kAmpMaxBins fits 16 bits)
    double* mult = nullptr;         // [nb] modes per bin
    double hyper[kAmpHyper] = {};   // host copy
    double* d_hyper = nullptr;      // [kAmpHyper]
    // state of the last forward evaluation
    float* theta = nullptr;         // [ntheta] copy of the argument
    double* ab = nullptr;           // [nb] A_b
    double* wn = nullptr;           // [nb] mult_b a_b^2 / S
    float* abf = nullptr;           // [nb] A_b rounded once (what the image-sized passes gather)
    float* dabf = nullptr;          // [nb] tangent dA_b
    double* gbin = nullptr;         // [nb] bin sums of an adjoint image
    double* work = nullptr;         // [4 nb] scratch of the scans
    double* sc = nullptr;           // [8] fluct, slope, flex, asp, zm, S
    float* xi = nullptr;            // [ny][nx] copy of the excitations of the joint position
    bool have_theta = false, have_xi = false;
    int ntheta() const { return kAmpScalars + 2 * (nb - 2); }
};

// ---- inverse-gamma point-source pixels (reading R18) ----
constexpr int kMaxPoints = 1024;
struct PointSources {
    int n = 0;
    double alpha = 0.0, q = 0.0;
    int* idx = nullptr;             // [n] position in the TRANSPOSED sky arrays: x ny + y
    float* xi = nullptr;            // [n] latent values of the current position (zeros until a joint call sets them)
    float* dv = nullptr;            // [n] tangent input of the metric (joint calls)
    float* out = nullptr;           // [n] gradient / metric output of the point latents
    double* flux = nullptr;         // [n] F^-1(Phi(xi))
    double* dflux = nullptr;        // [n] d flux / d xi
    double* sdiff = nullptr;        // [n] diffuse sky at the pixel
    double* stot = nullptr;         // [n] diffuse + flux
    bool in_sky = false;            // the cached sky contains the fluxes
};
// flux, dflux from p.xi
int launch_points_flux(cudaStream_t st, const PointSources& p);
// sky[idx] += flux, remembering the diffuse and the total value  (sky: transposed [nx][ny])
int launch_points_add(cudaStream_t st, const PointSources& p, float* sky);
// the fused passes multiply by the TOTAL sky; at a point-source pixel the Jacobian of the diffuse part is the diffuse sky
// and the point latent enters with dflux:  lin[idx] <- (sdiff lin[idx] + dflux dv) / stot   (dv may be null: 0)
int launch_points_pre(cudaStream_t st, const PointSources& p, float* lin, const float* dv);
// acc holds stot . c at the pixel:  out = sign dflux c (+ add);  acc[idx] <- sdiff c;  energy_acc (may be null) += 1/2 |add|^2
int launch_points_post(cudaStream_t st, const PointSources& p, float* acc, const float* add, float* out, double sign,
                       double* energy_acc);

int launch_amp_bins(cudaStream_t st, const AmpModel& m);
// theta -> A_b (and the state kept for the derivatives)
int launch_amp_forward(cudaStream_t st, const AmpModel& m);
// dA_b of dtheta at the stored theta -> m.dabf
int launch_amp_tangent(cudaStream_t st, const AmpModel& m, const float* dtheta);
// g_theta (+ theta_add if non-null) from the bin sums m.gbin; energy_acc (device double, may be null) += 1/2 |theta_add|^2
int launch_amp_adjoint(cudaStream_t st, const AmpModel& m, const float* theta_add, float* g_theta, double* energy_acc);
// out[pix] = table[pindex[pix]]
int launch_amp_gather(cudaStream_t st, const AmpModel& m, const float* table, float* out);
// m.gbin = bin sums of img (zeroed first)
int launch_amp_bin_reduce(cudaStream_t st, const AmpModel& m, const float* img);
// u = A . dxi + dA . xi   (A, dA gathered from the bin tables)
int launch_joint_prologue(cudaStream_t st, const AmpModel& m, const float* dxi, const float* xi, float* u);
// out_xi = A . h (+ add);  m.gbin = bin sums of xi . h
int launch_joint_epilogue(cudaStream_t st, const AmpModel& m, const float* h, const float* xi, const float* add, float* out_xi);

}  // namespace frs
