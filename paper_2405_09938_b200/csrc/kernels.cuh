// Launch wrappers of the four hot-path kernels (implemented in the .cu files beside this header).
#pragma once
#include "heeps_common.cuh"
#include "surface.cuh"

namespace heeps {

// K1 -- facet kinematics (kinematics.cu).  One launch fills `n_rows` rows: with H = 1 row r is pulse
// first + r; with H > 1 row r is keyframe first + r, i.e. pulse min((first + r) H, P - 1), and the time
// derivatives are written too (surface.cuh).
struct KinematicsArgs {
    const double2 *xt;      // [Nw][nx]  A_w exp(j kx_w x_i)
    const double2 *yt;      // [Nw][ny]  exp(j (ky_w y_j + phase_w))
    const double2 *tt;      // [Nw][P]   exp(-j omega_w t_p)
    const float4 *wk;       // [Nw]      {kx, ky, kx/|k|, ky/|k|}
    // Heterogeneous surface (eq. (1), (2)): nodes_x > 0 -- every table above (and omega) carries a leading
    // [nodes_y * nodes_x] dimension, one homogeneous tile T2L per node of a lattice of step node_spacing anchored at
    // the rest position of facet (0, 0); a facet blends the four corner tiles of its cell with the weights of eq. (2).
    int32_t nodes_x, nodes_y;
    double node_spacing;
    int32_t chunks_x, chunks_y;   // set by launch_kinematics: blocks per cell
    int32_t n_pulses_total; // P (row stride of tt)
    double *z;              // [n_pl][F]            surface height above centre_z
    float2 *slope;          // [n_pl][F] or null    grad z
    double2 *dxy;           // [n_pl][F] or null    CWM horizontal displacement
    int32_t H;              // keyframe spacing in pulses (1 = every pulse)
    const double *omega;    // [Nw] (H > 1)
    float *ztt;             // or null: second time derivative of the height [n_rows][F] (H > 1, no CWM), and with it
    float2 *slope_t;        //          the time derivative of the slopes [n_rows][F] (when slope is given)
    double *zt;             // time derivatives (H > 1): [n_rows][F]
    double2 *dxy_t;         // or null
};
cudaError_t launch_kinematics(const DevParams &prm, const KinematicsArgs &a, int first, int n_rows, cudaStream_t s);
int kinematics_coarse_row_slots(int n_rows);   // row slots a coarse-keyframe launch of n_rows pays for (kinematics.cu)
// K1b -- keyframe rows at spacing H interpolated from K1's coarse rows at spacing H1 (kinematics.cu).
struct SurfaceRefineArgs {
    const double *zc, *ztc;      // coarse rows [n_rows1][F]: height, its rate
    const float *zttc;           //                            its second time derivative
    const float2 *slopec, *slope_tc;   // or null: slopes and their rate
    double *z, *zt;              // out [n_rows][F]
    float2 *slope;               // out, or null
    const PulseConst *pulses;    // pulse times
    int64_t n_facets;
    int32_t H, H1, first, n_rows, first1, n_pulses_total;   // output row r = keyframe first + r (spacing H); coarse row 0 = coarse keyframe first1
};
cudaError_t launch_surface_refine(const SurfaceRefineArgs &a, cudaStream_t s);
cudaError_t launch_surface_slope(const DevParams &prm, const SurfaceArgs &sa, const PulseConst *pulses, int p,
                                 float2 *out, cudaStream_t s);

// K2 -- geometry, gains, amplitude, cull, tile bucketing (geometry.cu).
struct GeometryArgs {
    const PulseConst *pulses;   // [P]
    SurfaceArgs surf;           // from K1
    const float *sigma0;        // [F] or null
    const float2 *current;      // [F] or null
    const float2 *xi;           // [F]   complex speckle (debug outputs only)
    const uint2 *xi_polar;      // [F]   {|xi| as float bits, arg(xi) in 2^-32 turns}; [n_pl][F] with xi_pulse_stride = F
    int64_t xi_pulse_stride;    // 0: static speckle; F: time-dependent speckle, one row per pulse of the batch
    Rec *recs;                  // [C][n_pl][n_tiles][tile_cap]
    TileInfo *tinfo;            // [n_pl][n_tiles]
    TileSpan *tspan;            // [C][n_pl][n_tiles]
    unsigned long long *counters;  // [2]: kept facet-echoes, facet-samples (in-window, clipped to [0,Ns))
    // optional per-facet debug outputs (spatial order, single pulse): any may be null
    double *dbg_pos, *dbg_tau, *dbg_gtx, *dbg_grx, *dbg_amp;
    int32_t *dbg_keep;
    const double *carrier_frac_t0;  // [P] frac(f0 t0[p]) (debug amp only)
};
cudaError_t launch_geometry(const DevParams &prm, const GeometryArgs &a, int p0, int n_pl, cudaStream_t s);

// K3 -- echo accumulation, direct form (accumulate.cu).
struct AccumulateArgs {
    const Rec *recs;
    const TileInfo *tinfo;
    const TileSpan *tspan;
    double2 *acc;               // [C][n_pl][Ns] complex128 accumulators (zeroed by the caller)
    int block_threads;          // (warp groups) x warps_per_span x 32
    int samples_per_thread;     // R: a lane owns R consecutive samples of a record's window
    int warps_per_span;         // warps that together cover one window (32 R warps_per_span >= ceil(T fs))
    int span_cap;               // entries of each warp's shared-memory span array
    size_t smem_bytes;          // dynamic shared memory of the launch
};
struct AccumulatePlan {
    int block_threads, samples_per_thread, warps_per_span, span_cap;
    size_t smem_bytes;
};
// Launch shape from the replica length and the expected delay spread of a spatial tile [samples].
AccumulatePlan accumulate_plan(const DevParams &prm, double tile_spread_samples);
cudaError_t launch_accumulate(const DevParams &prm, const AccumulateArgs &a, int n_pl, cudaStream_t s);

// K4 -- finalize (finalize.cu): out = acc * exp(j 2 pi kappa (n-n_mid)^2) * exp(-j 2 pi f0 t0[p]) -> complex64
struct FinalizeArgs {
    const double2 *acc;         // [C][n_pl][Ns]
    const double2 *chirp_n;     // [Ns]  exp(j 2 pi kappa (n - n_mid)^2)
    const double2 *carrier_p;   // [P]   exp(-j 2 pi f0 t0[p])
    float2 *out;                // [C][n_out_pulses][Ns]
    int32_t n_out_pulses;       // pulse stride of `out`
    int32_t out_pulse0;         // index in `out` of the batch's first pulse
};
cudaError_t launch_finalize(const DevParams &prm, const FinalizeArgs &a, int p0, int n_pl, cudaStream_t s);

// Speckle from seed (G14): xi[f] = circular complex Gaussian, variance 1/2 per part, Philox4x32-10
// keyed by seed, counter = facet index, Box-Muller.
cudaError_t launch_speckle_from_seed(float2 *xi, int64_t n_facets, uint64_t seed, cudaStream_t s);
// xi -> {|xi|, arg(xi)} so that K2 can fold the speckle phase into the fixed-point phase word.
cudaError_t launch_speckle_polar(const float2 *xi, uint2 *xi_polar, int64_t n_facets, cudaStream_t s);

// Time-dependent speckle (speckle.cu; eq. (7), (10)): polar speckle of every facet at
// every pulse of a batch.
struct SpeckleAr1Args {
    const float2 *xi;              // [F]  R(0) + i I(0)
    float2 *state;                 // [F]  AR(1) state: read when `resume` (state after pulse p0 - 1), written on exit
    uint2 *polar;                  // [n_pl][F]  {|s|, arg s in 2^-32 turns} (Doppler factor included)
    const float2 *beta_g;          // [P]  {beta_q, sqrt(1 - beta_q^2)}, beta_q = exp(-(t_q - t_{q-1}) / tau_s); [0] unused
    const uint32_t *doppler_turns; // [P]  frac(f_s t_p) in 2^-32 turns
    int64_t n_facets;
    uint64_t seed;
    int32_t p0, n_pl, resume;
};
cudaError_t launch_speckle_ar1(const SpeckleAr1Args &a, cudaStream_t s);

// ---- spectral path (moments.cu, fftconv.cu) ----
constexpr int kMomentOrder = 8;   // Kt Chebyshev moments per range slice (truncation ~ J_8(pi B / 2 fs) ~ 1e-6)

// K2s -- geometry, gains, amplitude, cull, range-slice moments (moments.cu).
struct MomentArgs {
    const PulseConst *pulses;   // [P]
    SurfaceArgs surf;           // from K1
    const float *sigma0;        // [F] or null
    const float2 *current;      // [F] or null
    const uint2 *xi_polar;      // [F], or [n_pl][F] with xi_pulse_stride = F (time-dependent speckle)
    int64_t xi_pulse_stride;
    float2 *mom;                // [C][n_pl][Kt][nb_pad] complex moments, slice b at index b + L - 1 (zeroed by the caller)
    int32_t nb_pad;             // row stride (>= Ns + L - 1)
    int32_t span_cap;           // slices of a tile's shared-memory window
    int32_t replica;            // L = T fs (integer on this path)
    unsigned long long *counters;
    // K2k only, may be null: occupied slice range [band_lo, band_hi) of every vector [C][n_pl], by atomicMin / atomicMax
    // (the caller presets lo to a large and hi to a small value); lets K3s transform only the band (fftconv.cu)
    int32_t *band_lo, *band_hi;
    // K2k only, debug (sim_debug_echoes), all null in normal operation: what the kernel computes for the facet-echoes of
    // pulse dbg_pulse -- slice b [C][F], sub-slice position eps [C][F], complex weight [C][F] (before the reference phase
    // of the pulse), keep [F]
    int32_t *dbg_slice;
    float *dbg_eps;
    float2 *dbg_w;
    int32_t *dbg_keep;
    int32_t dbg_pulse;
};
size_t moments_smem_bytes(const DevParams &prm, int span_cap);
cudaError_t launch_moments(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, cudaStream_t s);

// K2k -- the same moments with the geometry evaluated exactly only at the kinematics keyframes and
// interpolated between (moments_keyframed.cu).  Needs surf.H in [2, kMaxKeyPulses - 1], C <= kMaxKeyChannels,
// series_channels; sim_create verifies the interpolation bounds on the host before choosing it.
constexpr int kMaxKeyChannels = 4;
constexpr int kMaxKeyPulses = 66;
size_t moments_keyframed_smem_bytes(const DevParams &prm, int span_cap);
bool moments_keyframed_fits(const DevParams &prm, int span_cap);
cudaError_t launch_moments_keyframed(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, cudaStream_t s);

// K3s -- convolution of the moments with the waveform kernels + finalize (fftconv.cu).
struct FftConvArgs {
    const float2 *mom;          // [C][n_pl][Kt][nb_pad]
    const float2 *cspec;        // [Kt][nfft]  FFT(c_k)/nfft in the forward transform's output order
    const float2 *tw;           // [nfft]      exp(-2 pi i k / nfft)
    const double2 *carrier_p;   // [P]         exp(-j 2 pi f0 t0[p])
    float2 *out;                // [C][n_out_pulses][Ns]
    int32_t n_out_pulses, out_pulse0;
    int32_t nfft;               // power of two, 256..16384, >= Ns + L - 1
    int32_t nb;                 // Ns + L - 1 valid slices
    int32_t nb_pad;
    int32_t replica;            // L
    // Band transform (optional, nfft2 = 0: off).  A vector whose occupied slices [band_lo, band_hi) satisfy
    // band_hi - band_lo + L - 1 <= nfft2 is convolved with an nfft2-point transform of the band alone (its echoes span a
    // fraction of the window: ATI 450 of 5295 slices), the others with the full nfft-point one.
    const int32_t *band_lo, *band_hi;   // [C][n_pl] from K2k
    const float2 *cspec2;       // [Kt][nfft2]
    const float2 *tw2;          // [nfft2]
    int32_t nfft2;
};
cudaError_t launch_fftconv(const DevParams &prm, const FftConvArgs &a, int p0, int n_pl, cudaStream_t s);
// cspec[k] = FFT(zero-padded ck[k][0..L)) / nfft for k < Kt (run once at sim_create).
cudaError_t launch_kernel_spectra(int nfft, const float2 *ck, int replica, const float2 *tw, float2 *cspec,
                                  cudaStream_t s);

}  // namespace heeps
