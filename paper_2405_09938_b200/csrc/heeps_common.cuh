// Shared device-side data layout of the raw-data generator kernels (K1..K4).
// Nothing here is shared with oracle/ (the oracle is an independent C file).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace heeps {

constexpr int kMaxChannels = 8;
constexpr double kC0 = 299792458.0;

// Per-pulse constants, computed on the host in fp64 at sim_create (stop-and-go, G9).
struct PulseConst {
    double t;                    // t_pulse[p]
    double r0;                   // c0 * t0[p]: bistatic path length of sample 0
    double tx_pos[3];
    double tx_a[3], tx_e[3];     // Tx azimuth / elevation axes
    double rx_a[3], rx_e[3];
    double rx_ref[3];            // un-offset Rx phase centre (cull reference, G6)
    double rx_pos[kMaxChannels][3];   // P_rx + o_c * v_rx/|v_rx|   (G8)
    double rx_vhat[3];           // v_rx/|v_rx|
    double rx_va, rx_ve;         // v^ . azimuth axis, v^ . elevation axis (Rx frame)
    double ch_off[kMaxChannels]; // o_c
    double tx_vel[3], rx_vel[3]; // platform velocities (keyframed geometry: d/dt of the path length)
};

// One surviving facet-echo as the accumulation kernel consumes it (32 B, 16 B aligned).
// Phase of sample n in turns:  phi + beta*(n - n_mid)  [+ kappa (n-n_mid)^2 applied in K4],
// in 32-bit fixed point (2^-32 turn); valid for n in [b, e).
// K2 adds a per-(tile, pulse, channel) frequency shift beta_s to every record of a tile so that the
// shifted tone frequency sits near a quarter cycle per sample (three-term recurrence best conditioned);
// K3 accumulates in that rotating frame and removes exp(j 2 pi beta_s (n - n_mid)) once per tile and sample.
struct __align__(16) Rec {
    uint32_t phi;                // frac(-dR/lambda + kappa c'^2 + arg(A~)/2pi) * 2^32 + bias (geometry.cu kPhiBias);
                                 // c' = echo centre - n_mid [samples], A~ = a_f G_tx G_rx,c
    uint32_t beta;               // frac(-2 kappa c' + beta_s) * 2^32
    float mag;                   // |A~|
    float wr;                    // Re exp(j 2 pi beta): one-sample phase step (shifted frame)
    float wi;                    // Im exp(j 2 pi beta)
    uint32_t flags;              // 0: three-term recurrence is well conditioned; 1: use the rotation
    int32_t b, e;                // in-window samples [b, e): b = ceil(nu), e = ceil(nu + T fs)
};
static_assert(sizeof(Rec) == 32, "Rec must be 32 bytes");

struct TileInfo {               // per (pulse-in-batch, tile)
    int32_t nrec;               // surviving facets (same for every channel)
};
struct __align__(16) TileSpan {  // per (channel, pulse-in-batch, tile)
    int32_t bmin, bmax_end;     // min b and max e over the tile's records
    uint32_t shift;             // beta_s in 2^-32 turns
    uint32_t pad;
};

// Antenna pattern as a complex u-v grid: tab[nv][nu] over the direction cosines
// u = r^ . azimuth axis, v = r^ . elevation axis; node k of u sits at u0 + k / su.  tab == nullptr: analytic sinc aperture.
struct PatternLut {
    const float2 *tab;
    int32_t nu, nv;
    double u0, su, v0, sv;
};

// Scalars every kernel needs.
struct DevParams {
    // grid / tiling
    int32_t nx, ny, tile, tiles_x, tiles_y, n_tiles, tile_cap;
    double spacing, cx, cy, cz;
    // instrument
    int32_t n_samples, n_channels, n_mid;
    double inv_lambda;           // f0/c0
    double fs_over_c0;           // samples per metre of bistatic path
    double kappa;                // K/(2 fs^2) turns per sample^2
    double half_len;             // T*fs/2 [samples]
    double len;                  // T*fs [samples]
    double ap_tx_a, ap_tx_e, ap_rx_a, ap_rx_e;   // aperture/lambda
    float cull_thr;              // 10^(dB/20) or 0
    // scene
    int32_t n_waves, choppy, tilt, has_sigma0, has_current;
    double sigma0_uniform, look_x, look_y, cur_ux, cur_uy;
    int32_t series_channels;     // receive-channel legs by series about the un-offset phase centre (geometry_common.cuh)
    int32_t lut_any;             // some antenna pattern is tabulated: gains are complex (geometry_common.cuh)
    PatternLut lut[2];           // [0] Tx, [1] Rx
    // keyframed geometry (moments_keyframed.cu): f0 / fs [turns of carrier per range slice] in units of 2^-48, split
    // into two 32-bit words, and the constant phase frac((2^15 - T fs / 2) f0 / fs) in 2^-32 turns
    uint32_t ratio_hi, ratio_lo, phase_bias32;
    // sheared tiles of K2k: k2k_h lines of k2k_w facets (k2k_w a power of two, k2k_w k2k_h = tile_cap); line b displaced by
    // rint(k2k_shear b) facets along the line; axis 0: lines = grid rows, 1: lines = grid columns; k2k_a0 = along-line
    // index of the first tile's first facet (<= 0); k2k_tiles_a tiles along a line, k2k_n_tiles in all
    int32_t k2k_w, k2k_h, k2k_cap, k2k_axis, k2k_a0, k2k_tiles_a, k2k_n_tiles;   // k2k_cap = k2k_w k2k_h facets per tile
    double k2k_shear;
};

}  // namespace heeps
