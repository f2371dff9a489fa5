// Host runtime + C ABI (include/heeps_sim.h) of the raw-data generator.
// Owns the device tables and the per-batch workspace, and sequences K1..K4 per pulse batch on
// the caller's stream with no host synchronisation inside sim_generate.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <new>
#include <atomic>
#include <string>
#include <thread>
#include <vector>

#include "../../include/heeps_sim.h"
#include "kernels.cuh"

using namespace heeps;

namespace {

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; }
        if (ok && prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    cudaError_t alloc(size_t count)
    {
        release();
        if (count == 0) return cudaSuccess;
        cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&p), count * sizeof(T));
        if (e == cudaSuccess) n = count; else p = nullptr;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; n = 0; }
};

}  // namespace

struct sim_handle {
    int device = 0;
    DevParams prm{};
    int n_pulses = 0;
    int64_t n_facets = 0;
    double chirp_rate = 0, chirp_len = 0, fs = 0;
    int pulses_per_batch = 1;
    AccumulatePlan accum{};              // K3 launch shape
    bool need_slope = false;
    bool spectral = false;               // accumulate_mode resolved at sim_create
    int nfft = 0, nb = 0, nb_pad = 0, replica = 0, span_cap_m = 0, span_cap_k = 0;   // slice window of a tile: K2s, K2k

    // tables
    DevBuf<double2> xt, yt, tt, chirp_n, carrier_p;
    DevBuf<float4> wk;
    DevBuf<double> carrier_frac;
    DevBuf<PulseConst> pulses;
    // maps
    DevBuf<float> sigma0;
    DevBuf<float2> current, xi;
    DevBuf<uint2> xi_polar;              // {|xi|, arg xi in 2^-32 turns}, derived from xi on the device
    DevBuf<float2> pattern[2];           // tabulated antenna patterns [nv][nu] (Tx, Rx), empty = analytic aperture
    // time-dependent speckle (speckle.cu; sim_scene.speckle_tau_s > 0)
    bool speckle_ar1 = false;
    uint64_t seed = 0;
    DevBuf<float2> xi_state, beta_g;     // AR(1) state after pulse xi_state_pulse; per-pulse {beta, sqrt(1 - beta^2)}
    DevBuf<uint32_t> doppler_turns;      // frac(f_s t_p) in 2^-32 turns
    DevBuf<uint2> xi_t;                  // [pulses_per_batch][F] polar speckle of the batch
    int xi_state_pulse = -1;
    float cur_lo[2] = {0.f, 0.f}, cur_hi[2] = {0.f, 0.f};   // bounding box of the current map at sim_create (widened by 25 %)
    // workspace
    DevBuf<double> z, zt, omega;
    DevBuf<float2> slope, slope_t;
    DevBuf<double2> dxy, dxy_t;
    int key_H = 1;                       // keyframe spacing of the kinematics (1 = every pulse)
    int key_H1 = 0;                      // > 0: K1 runs at this coarser spacing (a multiple of key_H) for the keyframed geometry kernel
    DevBuf<double> zc, ztc;              // K1's coarse keyframe rows (spacing key_H1): height, rate,
    DevBuf<float> zttc;                  //   second time derivative,
    DevBuf<float2> slopec, slope_tc;     //   slopes and their rate
    int nodes_x = 0, nodes_y = 0;        // heterogeneous surface: node lattice of the wave tables (0 = homogeneous)
    double node_spacing = 0;
    bool geo_keyframed = false;          // spectral path: ranges / gains interpolated between keyframes (K2k)
    int surf_rows_cap = 0;               // rows of the surface buffers
    DevBuf<Rec> recs;
    DevBuf<TileInfo> tinfo;
    DevBuf<TileSpan> tspan;
    DevBuf<double2> acc;
    DevBuf<unsigned long long> counters;
    DevBuf<float2> out_staging;
    // spectral path
    DevBuf<float2> mom, cspec, tw, cspec2, tw2;
    DevBuf<int32_t> band;               // [2][C * pulses_per_batch]: occupied slice range of every vector (K2k -> K3s)
    int nfft2 = 0;                      // band transform size, 0 = off

    // sim_debug_echoes: set for the duration of that call
    int32_t *dbg_slice = nullptr, *dbg_keep = nullptr;
    float *dbg_eps = nullptr;
    float2 *dbg_w = nullptr;
    int dbg_pulse = -1;
    // bookkeeping
    sim_stats stats{};
    bool profiling = false;
    std::vector<cudaEvent_t> events;     // 5 per batch when profiling
    size_t events_used = 0;
    std::string cuda_err;
    // sim_generate_host: device->host copies of finished batches overlap the next batch's kernels
    cudaStream_t copy_stream = nullptr;
    cudaStream_t aux_stream = nullptr;  // zeroes the moment rows while K1 runs
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    std::vector<cudaEvent_t> copy_events;

    ~sim_handle()
    {
        for (auto e : events) cudaEventDestroy(e);
        for (auto e : copy_events) cudaEventDestroy(e);
        if (copy_stream) cudaStreamDestroy(copy_stream);
        if (ev_fork) cudaEventDestroy(ev_fork);
        if (ev_join) cudaEventDestroy(ev_join);
        if (aux_stream) cudaStreamDestroy(aux_stream);
    }
};

namespace {

int fail_cuda(sim_handle *h, cudaError_t e, const char *what)
{
    if (h) {
        h->cuda_err = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
    }
    cudaGetLastError();   // clear the sticky-less error state
    return (e == cudaErrorMemoryAllocation) ? SIM_ENOMEM : SIM_ECUDA;
}

#define CK(h, call)                                                   \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return fail_cuda((h), e__, #call);    \
    } while (0)

// The wave tables of the scene: one homogeneous table, or one table per node of the heterogeneous lattice
// (sim_scene.wave_nodes_x > 0).  Entry (node, w) sits at index node * n_waves + w.
struct WaveView {
    int n_nodes, n_waves;
    const double *kx, *ky, *amp, *omega, *phase;
    bool hetero;
};
WaveView wave_view(const sim_scene *sc)
{
    if (sc->wave_nodes_x > 0)
        return {sc->wave_nodes_x * sc->wave_nodes_y, sc->n_waves, sc->node_kx, sc->node_ky, sc->node_amp, sc->node_omega,
                sc->node_phase, true};
    return {1, sc->n_waves, sc->kx, sc->ky, sc->amp, sc->omega, sc->phase, false};
}

bool finite_all(const double *p, size_t n)
{
    for (size_t k = 0; k < n; ++k) if (!std::isfinite(p[k])) return false;
    return true;
}

// Every value finite and, interleaved pairs (k & 1), inside [lo[k & 1], hi[k & 1]]: the scan of the per-facet maps
// (hundreds of megabytes on the large configurations, on the end-to-end path of sim_update_scene).  Branch-free inner
// loop (the exponent test on the bits, comparisons OR-ed into a mask), a few host threads for large maps: 336 MB in
// ~10 ms where the loop of std::isfinite with early exit took ~90 ms.
bool floats_ok(const float *p, size_t n, const float lo[2], const float hi[2])
{
    auto scan = [&](size_t b, size_t e) -> bool {        // [b, e), b even
        uint32_t bad = 0;
        const float l0 = lo[0], l1 = lo[1], h0 = hi[0], h1 = hi[1];
        size_t k = b;
        for (; k + 1 < e; k += 2) {
            uint32_t u0, u1;
            std::memcpy(&u0, p + k, 4); std::memcpy(&u1, p + k + 1, 4);
            bad |= (uint32_t)((u0 & 0x7f800000u) == 0x7f800000u) | (uint32_t)((u1 & 0x7f800000u) == 0x7f800000u);
            bad |= (uint32_t)(p[k] < l0) | (uint32_t)(p[k] > h0) | (uint32_t)(p[k + 1] < l1) | (uint32_t)(p[k + 1] > h1);
        }
        if (k < e) {
            uint32_t u0;
            std::memcpy(&u0, p + k, 4);
            bad |= (uint32_t)((u0 & 0x7f800000u) == 0x7f800000u) | (uint32_t)(p[k] < l0) | (uint32_t)(p[k] > h0);
        }
        return bad == 0;
    };
    const size_t kChunk = (size_t)1 << 22;
    if (n <= kChunk) return scan(0, n);
    const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
    const size_t n_chunks = (n + kChunk - 1) / kChunk;
    const unsigned n_thr = (unsigned)std::min<size_t>(std::min<unsigned>(hw, 8u), n_chunks);
    std::atomic<size_t> next{0};
    std::atomic<bool> ok{true};
    auto worker = [&]() {
        for (;;) {
            const size_t c = next.fetch_add(1);
            if (c >= n_chunks || !ok.load(std::memory_order_relaxed)) return;
            if (!scan(c * kChunk, std::min(n, (c + 1) * kChunk))) ok.store(false);
        }
    };
    std::vector<std::thread> pool;
    for (unsigned t = 1; t < n_thr; ++t) pool.emplace_back(worker);
    worker();
    for (auto &t : pool) t.join();
    return ok.load();
}

bool finite_all(const float *p, size_t n)
{
    const float lo[2] = {-3.4e38f, -3.4e38f}, hi[2] = {3.4e38f, 3.4e38f};
    return floats_ok(p, n, lo, hi);
}

bool frame_ok(const double *f)
{   // rows {b, a, e}: unit length, mutually orthogonal
    for (int r = 0; r < 3; ++r) {
        double n2 = f[3 * r] * f[3 * r] + f[3 * r + 1] * f[3 * r + 1] + f[3 * r + 2] * f[3 * r + 2];
        if (!(std::fabs(n2 - 1.0) < 1e-6)) return false;
        int q = (r + 1) % 3;
        double d = f[3 * r] * f[3 * q] + f[3 * r + 1] * f[3 * q + 1] + f[3 * r + 2] * f[3 * q + 2];
        if (!(std::fabs(d) < 1e-6)) return false;
    }
    return true;
}

int validate(const sim_instrument *in, const sim_geometry *g, const sim_scene *sc)
{
    if (!in || !g || !sc) return SIM_EINVAL;
    if (in->n_channels < 1 || in->n_channels > SIM_MAX_CHANNELS || !in->channel_offset_m) return SIM_EINVAL;
    if (in->n_samples < 1 || in->n_samples > (1 << 24)) return SIM_EINVAL;
    const double sc_in[] = {in->f0_hz, in->chirp_rate_hz_per_s, in->chirp_len_s, in->fs_hz, in->cull_two_way_db,
                            in->tx_aperture_m[0], in->tx_aperture_m[1], in->rx_aperture_m[0], in->rx_aperture_m[1]};
    if (!finite_all(sc_in, sizeof(sc_in) / sizeof(double))) return SIM_EINVAL;
    if (!(in->f0_hz > 0) || !(in->chirp_len_s > 0) || !(in->fs_hz > 0)) return SIM_EINVAL;
    if (in->tx_aperture_m[0] < 0 || in->tx_aperture_m[1] < 0 || in->rx_aperture_m[0] < 0 || in->rx_aperture_m[1] < 0)
        return SIM_EINVAL;
    if (!(in->chirp_len_s * in->fs_hz < (double)(1 << 22))) return SIM_EINVAL;
    if (!finite_all(in->channel_offset_m, in->n_channels)) return SIM_EINVAL;
    {   // tabulated antenna patterns: >= 2 x 2 nodes over an increasing, finite u-v range, finite values
        const float *tab[2] = {in->tx_pattern, in->rx_pattern};
        const int32_t nu[2] = {in->tx_pattern_nu, in->rx_pattern_nu}, nv[2] = {in->tx_pattern_nv, in->rx_pattern_nv};
        const double *ur[2] = {in->tx_pattern_u, in->rx_pattern_u}, *vr[2] = {in->tx_pattern_v, in->rx_pattern_v};
        for (int k = 0; k < 2; ++k) {
            if (!tab[k]) continue;
            if (nu[k] < 2 || nv[k] < 2 || (int64_t)nu[k] * nv[k] > ((int64_t)1 << 28)) return SIM_EINVAL;
            if (!finite_all(ur[k], 2) || !finite_all(vr[k], 2) || !(ur[k][1] > ur[k][0]) || !(vr[k][1] > vr[k][0]))
                return SIM_EINVAL;
            const size_t n = (size_t)nu[k] * nv[k] * 2;
            for (size_t i = 0; i < n; ++i) if (!std::isfinite(tab[k][i])) return SIM_EINVAL;
        }
    }
    if (g->n_pulses < 1) return SIM_EINVAL;
    if (!g->t_pulse_s || !g->tx_pos_m || !g->tx_vel_mps || !g->rx_pos_m || !g->rx_vel_mps || !g->tx_frame ||
        !g->rx_frame || !g->t0_s)
        return SIM_EINVAL;
    const size_t P = g->n_pulses;
    if (!finite_all(g->t_pulse_s, P) || !finite_all(g->t0_s, P) || !finite_all(g->tx_pos_m, 3 * P) ||
        !finite_all(g->rx_pos_m, 3 * P) || !finite_all(g->tx_vel_mps, 3 * P) || !finite_all(g->rx_vel_mps, 3 * P) ||
        !finite_all(g->tx_frame, 9 * P) || !finite_all(g->rx_frame, 9 * P))
        return SIM_EINVAL;
    for (size_t p = 0; p < P; ++p) {
        if (!frame_ok(g->tx_frame + 9 * p) || !frame_ok(g->rx_frame + 9 * p)) return SIM_EINVAL;
        const double *v = g->rx_vel_mps + 3 * p;
        if (!(v[0] * v[0] + v[1] * v[1] + v[2] * v[2] > 0)) return SIM_EINVAL;
    }
    if (sc->nx < 1 || sc->ny < 1 || (int64_t)sc->nx * sc->ny > ((int64_t)1 << 31)) return SIM_EINVAL;
    if (!(sc->spacing_m > 0) || !std::isfinite(sc->spacing_m) || !finite_all(sc->centre_m, 3)) return SIM_EINVAL;
    if (sc->n_waves < 0 || sc->n_waves > 4096) return SIM_EINVAL;
    if (sc->wave_nodes_x < 0 || sc->wave_nodes_y < 0) return SIM_EINVAL;
    if (sc->wave_nodes_x > 0) {
        // heterogeneous surface: a lattice of >= 2 x 2 nodes of step L anchored at facet (0, 0) that covers the grid
        if (sc->wave_nodes_x < 2 || sc->wave_nodes_y < 2 || sc->n_waves < 1) return SIM_EINVAL;
        if ((int64_t)sc->wave_nodes_x * sc->wave_nodes_y > (1 << 20)) return SIM_EINVAL;
        if (!(sc->wave_node_spacing_m > 0) || !std::isfinite(sc->wave_node_spacing_m)) return SIM_EINVAL;
        if (!sc->node_kx || !sc->node_ky || !sc->node_amp || !sc->node_omega || !sc->node_phase) return SIM_EINVAL;
        const double L = sc->wave_node_spacing_m * (1.0 + 1e-12);
        if ((sc->nx - 1) * sc->spacing_m > (sc->wave_nodes_x - 1) * L || (sc->ny - 1) * sc->spacing_m > (sc->wave_nodes_y - 1) * L)
            return SIM_EINVAL;
        const size_t n = (size_t)sc->wave_nodes_x * sc->wave_nodes_y * sc->n_waves;
        if (!finite_all(sc->node_kx, n) || !finite_all(sc->node_ky, n) || !finite_all(sc->node_amp, n) ||
            !finite_all(sc->node_omega, n) || !finite_all(sc->node_phase, n))
            return SIM_EINVAL;
    } else if (sc->n_waves > 0) {
        if (!sc->kx || !sc->ky || !sc->amp || !sc->omega || !sc->phase) return SIM_EINVAL;
        if (!finite_all(sc->kx, sc->n_waves) || !finite_all(sc->ky, sc->n_waves) || !finite_all(sc->amp, sc->n_waves) ||
            !finite_all(sc->omega, sc->n_waves) || !finite_all(sc->phase, sc->n_waves))
            return SIM_EINVAL;
    }
    if (!sc->sigma0_lin && !(sc->sigma0_uniform >= 0 && std::isfinite(sc->sigma0_uniform))) return SIM_EINVAL;
    {   // the per-facet maps: finite everywhere (a NaN current or sigma0 would poison whole tiles), sigma0 >= 0
        const size_t F = (size_t)sc->nx * sc->ny;
        if (sc->sigma0_lin) {
            const float lo[2] = {0.f, 0.f}, hi[2] = {3.4e38f, 3.4e38f};
            if (!floats_ok(sc->sigma0_lin, F, lo, hi)) return SIM_EINVAL;
        }
        if (sc->current_mps && !finite_all(sc->current_mps, 2 * F)) return SIM_EINVAL;
        if (sc->xi && !finite_all(sc->xi, 2 * F)) return SIM_EINVAL;
    }
    if (!finite_all(sc->look_dir, 2) || !finite_all(sc->current_uniform, 2)) return SIM_EINVAL;
    if (!std::isfinite(sc->speckle_tau_s) || !std::isfinite(sc->speckle_doppler_hz)) return SIM_EINVAL;
    if (sc->speckle_tau_s > 0)
        for (int p = 0; p + 1 < g->n_pulses; ++p) if (!(g->t_pulse_s[p + 1] >= g->t_pulse_s[p])) return SIM_EINVAL;
    return SIM_OK;
}

// Horizontal gradient magnitude bound of the bistatic path at the scene centre, mid dwell
// (flat surface): |d(r_t+r_r)/dx| + |d(r_t+r_r)/dy|, used only to size tiles and CTAs.
// Extent of the scene in bistatic path length [m] at a pulse, largest over the dwell and the channels: 9 x 9 lattice of
// rest positions (the path length is convex over the rectangle: its maximum sits at a corner, the lattice bounds its
// minimum to a cell) plus the vertical excursion of the waves on both legs.  Sizes the band transform; not a guarantee.
double scene_slice_extent(const sim_instrument *in, const sim_geometry *g, const sim_scene *sc, double wave_sum)
{
    double worst = 0;
    const int P = g->n_pulses, step = std::max(1, P / 64);
    for (int p = 0; p < P; p = (p + step < P || p == P - 1) ? p + step : P - 1) {
        const double *tx = g->tx_pos_m + 3 * p, *rx = g->rx_pos_m + 3 * p, *rv = g->rx_vel_mps + 3 * p;
        const double vn = std::sqrt(rv[0] * rv[0] + rv[1] * rv[1] + rv[2] * rv[2]);
        const double tdrift = g->t_pulse_s[p];
        for (int c = 0; c < in->n_channels; ++c) {
            const double o = in->channel_offset_m[c];
            const double rc[3] = {rx[0] + o * rv[0] / vn, rx[1] + o * rv[1] / vn, rx[2] + o * rv[2] / vn};
            double lo = 1e300, hi = -1e300;
            for (int a = 0; a <= 8; ++a)
                for (int b = 0; b <= 8; ++b) {
                    const double x = sc->centre_m[0] + (a / 8.0 - 0.5) * (sc->nx - 1) * sc->spacing_m + sc->current_uniform[0] * tdrift;
                    const double y = sc->centre_m[1] + (b / 8.0 - 0.5) * (sc->ny - 1) * sc->spacing_m + sc->current_uniform[1] * tdrift;
                    const double z = sc->centre_m[2];
                    const double r = std::sqrt((x - tx[0]) * (x - tx[0]) + (y - tx[1]) * (y - tx[1]) + (z - tx[2]) * (z - tx[2])) +
                                     std::sqrt((x - rc[0]) * (x - rc[0]) + (y - rc[1]) * (y - rc[1]) + (z - rc[2]) * (z - rc[2]));
                    lo = std::min(lo, r); hi = std::max(hi, r);
                }
            worst = std::max(worst, hi - lo);
        }
    }
    return worst + 4.0 * wave_sum;
}

double path_gradient_l1(const sim_geometry *g, const sim_scene *sc)
{
    double worst = 0;
    const int P = g->n_pulses;
    const int picks[3] = {0, P / 2, P - 1};
    for (int q = 0; q < 3; ++q) {
        const double *tx = g->tx_pos_m + 3 * picks[q], *rx = g->rx_pos_m + 3 * picks[q];
        // evaluate at centre and the four scene corners
        for (int cx = -1; cx <= 1; ++cx)
            for (int cy = -1; cy <= 1; ++cy) {
                double x = sc->centre_m[0] + cx * 0.5 * sc->nx * sc->spacing_m;
                double y = sc->centre_m[1] + cy * 0.5 * sc->ny * sc->spacing_m;
                double z = sc->centre_m[2];
                double dt[3] = {x - tx[0], y - tx[1], z - tx[2]}, dr[3] = {x - rx[0], y - rx[1], z - rx[2]};
                double rt = std::sqrt(dt[0] * dt[0] + dt[1] * dt[1] + dt[2] * dt[2]);
                double rr = std::sqrt(dr[0] * dr[0] + dr[1] * dr[1] + dr[2] * dr[2]);
                double gx = dt[0] / rt + dr[0] / rr, gy = dt[1] / rt + dr[1] / rr;
                worst = std::max(worst, std::fabs(gx) + std::fabs(gy));
            }
    }
    return worst;
}

// Sheared tiles of the keyframed geometry kernel (moments_keyframed.cu): TH lines of TW facets, line b displaced by
// rint(shear b) facets, so that a tile is as narrow in range as its lines are.  From the path-length gradient (in range
// slices per facet step) at the scene centre, mid dwell, the shear that puts equal facets of all lines on one iso-range
// line; its worst-case extent over a 3 x 3 lattice of scene points and three pulses sizes the tile's slice window.  The
// shape with the smallest (tiles x (1 + extent / 16)) wins -- a displaced tiling has a few partly empty tiles per band.
struct ShearPlan {
    int w = 32, h = 32, axis = 0, a0 = 0, tiles_a = 1, tiles_b = 1;
    double shear = 0, extent = 0;
};
ShearPlan plan_sheared_tiles(const sim_geometry *g, const sim_scene *sc, double fsc, int tile_cap)
{
    const int P = g->n_pulses;
    const int picks[3] = {0, P / 2, P - 1};
    struct G2 { double gx, gy; };
    auto grad_at = [&](int p, double x, double y) {
        const double *tx = g->tx_pos_m + 3 * p, *rx = g->rx_pos_m + 3 * p;
        const double z = sc->centre_m[2];
        const double dt[3] = {x - tx[0], y - tx[1], z - tx[2]}, dr[3] = {x - rx[0], y - rx[1], z - rx[2]};
        const double rt = std::sqrt(dt[0] * dt[0] + dt[1] * dt[1] + dt[2] * dt[2]);
        const double rr = std::sqrt(dr[0] * dr[0] + dr[1] * dr[1] + dr[2] * dr[2]);
        return G2{(dt[0] / rt + dr[0] / rr) * sc->spacing_m * fsc, (dt[1] / rt + dr[1] / rr) * sc->spacing_m * fsc};
    };
    std::vector<G2> samples;
    for (int q = 0; q < 3; ++q)
        for (int cx = -1; cx <= 1; ++cx)
            for (int cy = -1; cy <= 1; ++cy)
                samples.push_back(grad_at(picks[q], sc->centre_m[0] + cx * 0.5 * (sc->nx - 1) * sc->spacing_m,
                                          sc->centre_m[1] + cy * 0.5 * (sc->ny - 1) * sc->spacing_m));
    const G2 c = grad_at(P / 2, sc->centre_m[0], sc->centre_m[1]);
    ShearPlan best;
    double best_cost = 1e300;
    for (int axis = 0; axis < 2; ++axis)
        for (int tw = 4; tw <= tile_cap / 2; tw <<= 1) {
            const int th = tile_cap / tw;
            if (tw * th != tile_cap) continue;
            const double ga = axis ? c.gy : c.gx, gb = axis ? c.gx : c.gy;
            const int na = axis ? sc->ny : sc->nx, nb = axis ? sc->nx : sc->ny;
            for (int use_shear = 0; use_shear < 2; ++use_shear) {
                double sh = 0;
                if (use_shear) {
                    if (std::fabs(ga) < 1e-9) continue;
                    sh = -gb / ga;
                    const double lim = std::min(4.0 * tw, 128.0) / th;      // at most four extra tiles per band
                    sh = std::max(-lim, std::min(lim, sh));
                }
                double ext = 0;
                for (const G2 &s2 : samples) {
                    const double sa = axis ? s2.gy : s2.gx, sb = axis ? s2.gx : s2.gy;
                    ext = std::max(ext, tw * std::fabs(sa) + th * std::fabs(sb + sa * sh) + std::fabs(sa));
                }
                int smin = 0, smax = 0;
                for (int b = 0; b < th; ++b) {
                    const int v = (int)std::nearbyint(sh * b);
                    smin = std::min(smin, v); smax = std::max(smax, v);
                }
                const int tiles_a = (na + (smax - smin) + tw - 1) / tw, tiles_b = (nb + th - 1) / th;
                const double cost = (double)tiles_a * tiles_b * (1.0 + ext / 16.0);
                if (cost < best_cost) {
                    best_cost = cost;
                    best.w = tw; best.h = th; best.axis = axis; best.a0 = -smax; best.tiles_a = tiles_a; best.tiles_b = tiles_b;
                    best.shear = sh; best.extent = ext;
                }
            }
        }
    return best;
}

// Rows of the surface buffers a batch [p0, p0 + n_pl) needs: its pulses (H = 1) or its keyframes.
void surface_rows(const sim_handle *h, int p0, int n_pl, int *first, int *rows, int spacing = 0)
{
    const int H = spacing > 0 ? spacing : h->key_H, P = h->n_pulses;
    if (H <= 1) { *first = p0; *rows = n_pl; return; }
    const int n_keys = (P - 1 + H - 1) / H + 1;
    const int j0 = std::min(p0 / H, n_keys - 2), j1 = std::min((p0 + n_pl - 1) / H, n_keys - 2) + 1;
    *first = j0; *rows = j1 - j0 + 1;
}

struct SurfBufs {
    double *z, *zt; float2 *slope, *slope_t; double2 *dxy, *dxy_t;
};

// Time-dependent speckle of the batch (speckle.cu): fills h->xi_t and returns the pointer / row stride the K2 kernels use.
int run_speckle(sim_handle *h, int p0, int n_pl, cudaStream_t s, const uint2 **polar, int64_t *stride)
{
    *polar = h->xi_polar.p; *stride = 0;
    if (!h->speckle_ar1) return SIM_OK;
    SpeckleAr1Args a{};
    a.xi = h->xi.p; a.state = h->xi_state.p; a.polar = h->xi_t.p; a.beta_g = h->beta_g.p;
    a.doppler_turns = h->doppler_turns.p; a.n_facets = h->n_facets; a.seed = h->seed;
    a.p0 = p0; a.n_pl = n_pl;
    a.resume = (p0 > 0 && h->xi_state_pulse == p0 - 1) ? 1 : 0;
    cudaError_t e = launch_speckle_ar1(a, s);
    if (e != cudaSuccess) return fail_cuda(h, e, "launch_speckle_ar1");
    h->xi_state_pulse = p0 + n_pl - 1;
    *polar = h->xi_t.p; *stride = h->n_facets;
    return SIM_OK;
}

// K1 for the batch; fills `sa` for K2.
// `coarse`: K1 runs at the coarser spacing key_H1 (with second derivatives) into the coarse buffers and K1b interpolates
// the rows at spacing key_H from them; what the geometry kernel sees is the same either way.
int run_kinematics(sim_handle *h, const SurfBufs &b, int p0, int n_pl, cudaStream_t s, SurfaceArgs *sa, bool coarse = false)
{
    int first = 0, rows = 0;
    surface_rows(h, p0, n_pl, &first, &rows);
    KinematicsArgs ka{};
    ka.xt = h->xt.p; ka.yt = h->yt.p; ka.tt = h->tt.p; ka.wk = h->wk.p; ka.n_pulses_total = h->n_pulses;
    ka.nodes_x = h->nodes_x; ka.nodes_y = h->nodes_y; ka.node_spacing = h->node_spacing;
    ka.z = b.z; ka.slope = b.slope; ka.dxy = b.dxy;
    ka.H = h->key_H; ka.omega = h->omega.p; ka.zt = b.zt; ka.dxy_t = b.dxy_t;
    if (coarse) {
        int first1 = 0, rows1 = 0;
        surface_rows(h, p0, n_pl, &first1, &rows1, h->key_H1);
        ka.z = h->zc.p; ka.zt = h->ztc.p; ka.ztt = h->zttc.p; ka.H = h->key_H1;
        ka.slope = b.slope ? h->slopec.p : nullptr; ka.slope_t = b.slope ? h->slope_tc.p : nullptr;
        cudaError_t e = launch_kinematics(h->prm, ka, first1, rows1, s);
        if (e != cudaSuccess) return fail_cuda(h, e, "launch_kinematics (coarse)");
        SurfaceRefineArgs ra{};
        ra.zc = h->zc.p; ra.ztc = h->ztc.p; ra.zttc = h->zttc.p; ra.slopec = ka.slope; ra.slope_tc = ka.slope_t;
        ra.z = b.z; ra.zt = b.zt; ra.slope = b.slope; ra.pulses = h->pulses.p; ra.n_facets = h->n_facets;
        ra.H = h->key_H; ra.H1 = h->key_H1; ra.first = first; ra.n_rows = rows; ra.first1 = first1; ra.n_pulses_total = h->n_pulses;
        e = launch_surface_refine(ra, s);
        if (e != cudaSuccess) return fail_cuda(h, e, "launch_surface_refine");
    } else {
        cudaError_t e = launch_kinematics(h->prm, ka, first, rows, s);
        if (e != cudaSuccess) return fail_cuda(h, e, "launch_kinematics");
    }
    sa->z = b.z; sa->zt = b.zt; sa->slope = b.slope; sa->slope_t = nullptr; sa->dxy = b.dxy; sa->dxy_t = b.dxy_t;
    sa->H = h->key_H; sa->key0 = first; sa->n_pulses_total = h->n_pulses;
    return SIM_OK;
}

// Keyframe spacing (surface.cuh): largest H <= 64 whose cubic-Hermite error bound sum_w A_w (omega_w h)^4 / 384 stays
// under kKeyframeHeightTol (9e-6 rad of carrier phase on the two legs, worst case with all components in phase; the same
// for the CWM displacement) and, with tilt modulation, whose linear-interpolation error of the slopes, 4 x the
// root-sum-square of A_w |k_w| (omega_w h)^2 / 8 over the components (random phases), stays under kKeyframeSlopeTol (the
// slopes only scale sigma0: measured 1.8e-5 of relative L2 on the Large configuration at H = 32); 1 when pulse times are
// not increasing.
constexpr double kKeyframeHeightTol = 4e-8, kKeyframeSlopeTol = 1.2e-4;

// Decoupled keyframes.  The geometry kernel needs the surface only at ITS keyframes (spacing H, bounded by its cubic path
// interpolant); K1 -- 15 % of a step at that spacing -- can run at a multiple R H of it when it also stores the second
// time derivative of the height and the rate of the slopes: between K1's keyframes the height is the QUINTIC Hermite
// interpolant (error <= sum_w A_w (omega_w h)^6 / 46080), its rate the derivative of that (error <= sum_w A_w omega_w
// (omega_w h)^5 / 1920, times the interval of the geometry kernel as a path error), the slopes the cubic one
// (<= sum_w A_w |k_w| (omega_w h)^4 / 384).  Largest R in {4, 2} within a quarter of the height bound (the geometry
// kernel's own cubic adds its part) and kCoarseSlopeTol on the slopes (they only scale sigma0; the linear interpolation
// between the geometry kernel's keyframes that follows is allowed kKeyframeSlopeTol = 1.2e-4); 0 = keep one spacing.
constexpr double kCoarseSlopeTol = 1e-5;
int choose_coarse_spacing(const sim_geometry *g, const sim_scene *sc, int H)
{
    const int P = g->n_pulses;
    const WaveView wv = wave_view(sc);
    for (int R = 4; R >= 2; R >>= 1) {
        const int H1 = R * H;
        if (H1 > P - 1) continue;
        double hmax = 0, hk = 0;
        for (int k = 0; k < P - 1; k += H1) hmax = std::max(hmax, g->t_pulse_s[std::min(k + H1, P - 1)] - g->t_pulse_s[k]);
        for (int k = 0; k < P - 1; k += H) hk = std::max(hk, g->t_pulse_s[std::min(k + H, P - 1)] - g->t_pulse_s[k]);
        double bz = 0, bv = 0, bs = 0;
        for (int n = 0; n < wv.n_nodes; ++n) {
            double z1 = 0, v1 = 0, s1 = 0;
            for (int w = 0; w < wv.n_waves; ++w) {
                const size_t k = (size_t)n * wv.n_waves + w;
                const double x = wv.omega[k] * hmax, a = std::fabs(wv.amp[k]);
                z1 += a * std::pow(x, 6) / 46080.0;
                v1 += a * wv.omega[k] * std::pow(x, 5) / 1920.0;
                s1 += a * std::hypot(wv.kx[k], wv.ky[k]) * std::pow(x, 4) / 384.0;
            }
            bz = std::max(bz, z1); bv = std::max(bv, v1); bs = std::max(bs, s1);
        }
        if (wv.hetero) { bz *= 2.0; bv *= 2.0; bs *= 2.0; }
        if (bz + 0.125 * hk * bv <= 0.25 * kKeyframeHeightTol && (!sc->tilt_modulation || bs <= kCoarseSlopeTol)) return H1;
    }
    return 0;
}

int choose_keyframe_spacing(const sim_geometry *g, const sim_scene *sc, int requested)
{
    const int P = g->n_pulses;
    if (requested == 1 || P < 4 || sc->n_waves == 0) return 1;
    for (int p = 0; p + 1 < P; ++p) if (!(g->t_pulse_s[p + 1] > g->t_pulse_s[p])) return 1;
    if (requested > 1) return std::min(requested, P - 1);
    for (int H = 64; H >= 2; H >>= 1) {
        if (H > P - 1) continue;
        double hmax = 0;
        for (int k = 0; k < P - 1; k += H) hmax = std::max(hmax, g->t_pulse_s[std::min(k + H, P - 1)] - g->t_pulse_s[k]);
        // heterogeneous surface: four tiles with weights that add to at most 2 (squares to 1): worst node, doubled
        const WaveView wv = wave_view(sc);
        double bound = 0, slope2 = 0;
        for (int n = 0; n < wv.n_nodes; ++n) {
            double b1 = 0, s2 = 0;
            for (int w = 0; w < wv.n_waves; ++w) {
                const size_t k = (size_t)n * wv.n_waves + w;
                const double x = wv.omega[k] * hmax;
                b1 += std::fabs(wv.amp[k]) * x * x * x * x / 384.0;
                const double sl = std::fabs(wv.amp[k]) * std::hypot(wv.kx[k], wv.ky[k]) * x * x / 8.0;
                s2 += sl * sl;
            }
            bound = std::max(bound, b1); slope2 = std::max(slope2, s2);
        }
        if (wv.hetero) bound *= 2.0;
        if (bound <= kKeyframeHeightTol && (!sc->tilt_modulation || 4.0 * std::sqrt(slope2) <= kKeyframeSlopeTol)) return H;
    }
    return 1;
}

// ---- guard of the keyframed geometry (moments_keyframed.cu) ----
// Evaluates, in long double on a 3 x 3 lattice of scene points (rest height, drifting with the uniform
// current), the three interpolants the kernel uses over every keyframe interval of spacing H -- Hermite path
// length, linear receive-channel path difference, cubic gain product with the finite-difference channel
// term -- against the exact geometry at EVERY pulse.  True iff all stay inside: path kGuardPathTol, gains kGuardGainTol
// (tabulated: kGuardGainTolLut); the scene points drift with the uniform current or, with a current map, with each corner
// of the bounding box of its values.
long double sincl_pi(long double x)
{
    if (x == 0.0L) return 1.0L;
    const long double a = 3.14159265358979323846264338327950288L * x;
    return sinl(a) / a;
}

typedef std::complex<long double> cld;

struct GuardEval {
    long double R, Rd, xat, xet, xar, xer, xao, xeo, dl[SIM_MAX_CHANNELS], gt, gr[SIM_MAX_CHANNELS];
    long double uat, uet, uar, uer, uao, ueo;          // the six sinc arguments as direction cosines
    cld gtc, grc[SIM_MAX_CHANNELS];                    // complex gains (tabulated patterns, reading G29; else (analytic, 0))
};

// Complex gain of antenna k (0 Tx, 1 Rx) at direction cosines (ua, ue): bilinear in the u-v table when there is one
// (zero outside the grid), else the analytic aperture pattern.
cld host_gain(const sim_instrument *in, int k, long double ua, long double ue)
{
    const float *tab = k ? in->rx_pattern : in->tx_pattern;
    if (!tab) {
        const long double lambda = (long double)kC0 / in->f0_hz;
        const double *ap = k ? in->rx_aperture_m : in->tx_aperture_m;
        return cld(sincl_pi(ap[0] / lambda * ua) * sincl_pi(ap[1] / lambda * ue), 0.0L);
    }
    const int nu = k ? in->rx_pattern_nu : in->tx_pattern_nu, nv = k ? in->rx_pattern_nv : in->tx_pattern_nv;
    const double *ur = k ? in->rx_pattern_u : in->tx_pattern_u, *vr = k ? in->rx_pattern_v : in->tx_pattern_v;
    const long double gu = (ua - ur[0]) * (nu - 1) / ((long double)ur[1] - ur[0]);
    const long double gv = (ue - vr[0]) * (nv - 1) / ((long double)vr[1] - vr[0]);
    if (!(gu >= 0 && gu <= nu - 1 && gv >= 0 && gv <= nv - 1)) return cld(0, 0);
    const int iu = std::min((int)gu, nu - 2), iv = std::min((int)gv, nv - 2);
    const long double fu = gu - iu, fv = gv - iv;
    auto node = [&](int a, int b) { const float *t = tab + 2 * ((size_t)(iv + b) * nu + iu + a); return cld(t[0], t[1]); };
    return (1 - fv) * ((1 - fu) * node(0, 0) + fu * node(1, 0)) + fv * ((1 - fu) * node(0, 1) + fu * node(1, 1));
}

// Largest |second difference| / 8 of a table along u plus along v: the distance between the bilinear interpolant and
// any smooth function through the nodes (h^2 |G''| / 8 per axis); and the largest |node|.  (0, 1) for an analytic antenna.
void table_roughness(const sim_instrument *in, int k, long double &delta, long double &gmax)
{
    const float *tab = k ? in->rx_pattern : in->tx_pattern;
    delta = 0; gmax = 1;
    if (!tab) return;
    const int nu = k ? in->rx_pattern_nu : in->tx_pattern_nu, nv = k ? in->rx_pattern_nv : in->tx_pattern_nv;
    auto node = [&](int a, int b) { const float *t = tab + 2 * ((size_t)b * nu + a); return std::complex<double>(t[0], t[1]); };
    double du = 0, dv = 0, gm = 0;
    for (int b = 0; b < nv; ++b)
        for (int a = 0; a < nu; ++a) {
            gm = std::max(gm, std::abs(node(a, b)));
            if (a > 0 && a + 1 < nu) du = std::max(du, std::abs(node(a - 1, b) - 2.0 * node(a, b) + node(a + 1, b)));
            if (b > 0 && b + 1 < nv) dv = std::max(dv, std::abs(node(a, b - 1) - 2.0 * node(a, b) + node(a, b + 1)));
        }
    delta = (du + dv) / 8; gmax = gm;
}

GuardEval guard_eval(const sim_instrument *in, const sim_geometry *g, int p, const long double pos[3],
                     const long double vel[3], long double o_fd)
{
    GuardEval o{};
    const long double lambda = (long double)kC0 / in->f0_hz;
    const double *tp = g->tx_pos_m + 3 * p, *rp = g->rx_pos_m + 3 * p, *tv = g->tx_vel_mps + 3 * p,
                 *rv = g->rx_vel_mps + 3 * p, *tf = g->tx_frame + 9 * p, *rf = g->rx_frame + 9 * p;
    long double vn = sqrtl((long double)rv[0] * rv[0] + (long double)rv[1] * rv[1] + (long double)rv[2] * rv[2]);
    long double dt[3], dr[3], rt = 0, rr = 0;
    for (int k = 0; k < 3; ++k) { dt[k] = pos[k] - tp[k]; dr[k] = pos[k] - rp[k]; rt += dt[k] * dt[k]; rr += dr[k] * dr[k]; }
    rt = sqrtl(rt); rr = sqrtl(rr);
    o.R = rt + rr;
    for (int k = 0; k < 3; ++k) o.Rd += dt[k] * (vel[k] - tv[k]) / rt + dr[k] * (vel[k] - rv[k]) / rr;
    auto args = [&](const long double d[3], long double r, const double *frame, const double ap[2], long double &xa,
                    long double &xe) {
        long double da = 0, de = 0;
        for (int k = 0; k < 3; ++k) { da += d[k] * frame[3 + k]; de += d[k] * frame[6 + k]; }
        xa = ap[0] / lambda * da / r; xe = ap[1] / lambda * de / r;
    };
    args(dt, rt, tf, in->tx_aperture_m, o.xat, o.xet);
    args(dr, rr, rf, in->rx_aperture_m, o.xar, o.xer);
    o.gt = sincl_pi(o.xat) * sincl_pi(o.xet);
    auto cosines = [&](const long double d[3], long double r, const double *frame, long double &ua, long double &ue) {
        ua = ue = 0;
        for (int k = 0; k < 3; ++k) { ua += d[k] * frame[3 + k]; ue += d[k] * frame[6 + k]; }
        ua /= r; ue /= r;
    };
    cosines(dt, rt, tf, o.uat, o.uet);
    cosines(dr, rr, rf, o.uar, o.uer);
    o.gtc = host_gain(in, 0, o.uat, o.uet);
    auto offset_leg = [&](long double off, long double &r_c, long double &xa, long double &xe, long double &ua,
                          long double &ue) {
        long double d[3]; r_c = 0;
        for (int k = 0; k < 3; ++k) { d[k] = pos[k] - (rp[k] + off * rv[k] / vn); r_c += d[k] * d[k]; }
        r_c = sqrtl(r_c);
        args(d, r_c, rf, in->rx_aperture_m, xa, xe);
        cosines(d, r_c, rf, ua, ue);
    };
    long double r_o;
    offset_leg(o_fd, r_o, o.xao, o.xeo, o.uao, o.ueo);
    for (int c = 0; c < in->n_channels; ++c) {
        long double r_c, xa, xe, ua, ue;
        offset_leg(in->channel_offset_m[c], r_c, xa, xe, ua, ue);
        o.dl[c] = r_c - rr;
        o.gr[c] = sincl_pi(xa) * sincl_pi(xe);
        o.grc[c] = host_gain(in, 1, ua, ue);
    }
    return o;
}

// Waveform kernels of the moment form (moments.cu header): with b = ceil(nu) the slice of a facet-echo, eps = b - nu its
// sub-slice position and y = 2 eps - 1, sample n = b + m of its replica is
//     g_m(y) = exp(j 2 pi kappa (m + (y + 1)/2 - L/2)^2),     y in [-1, 1],
// and c_k[m] are the Chebyshev coefficients of g_m in y (Gauss-Chebyshev quadrature on 64 nodes: exact to rounding
// for this entire function), so that  s[n] = sum_k sum_m c_k[m] M_k[n - m]  with the Chebyshev moments M_k of the
// slices.  Returns c_k for k < n_k ([n_k][L]) and max_m |c_k[m]| per k: the tail beyond Kt bounds the truncation.
void chebyshev_kernels(double kappa, int L, int n_k, std::vector<std::complex<double>> &ck, std::vector<double> &cmax)
{
    const int NQ = 64;
    ck.assign((size_t)n_k * L, std::complex<double>(0, 0));
    cmax.assign(n_k, 0.0);
    std::vector<double> cs((size_t)n_k * NQ), yq(NQ);
    for (int j = 0; j < NQ; ++j) {
        const double th = M_PI * (j + 0.5) / NQ;
        yq[j] = std::cos(th);
        for (int k = 0; k < n_k; ++k) cs[(size_t)k * NQ + j] = std::cos(k * th);
    }
    std::vector<std::complex<double>> gq(NQ);
    for (int m = 0; m < L; ++m) {
        for (int j = 0; j < NQ; ++j) {
            const long double u = (long double)m + 0.5L * ((long double)yq[j] + 1.0L) - 0.5L * (long double)L;
            long double turns = (long double)kappa * u * u;
            turns -= floorl(turns);
            gq[j] = std::complex<double>(std::cos(2.0 * M_PI * (double)turns), std::sin(2.0 * M_PI * (double)turns));
        }
        for (int k = 0; k < n_k; ++k) {
            std::complex<double> acc(0, 0);
            for (int j = 0; j < NQ; ++j) acc += gq[j] * cs[(size_t)k * NQ + j];
            acc *= (k ? 2.0 : 1.0) / NQ;
            ck[(size_t)k * L + m] = acc;
            cmax[k] = std::max(cmax[k], std::abs(acc));
        }
    }
}
constexpr double kMomentTruncationTol = 5e-6;    // sum over k >= Kt of max_m |c_k[m]| the spectral form accepts (bar: 1e-4)

// Tolerances of the guard: path 2e-8 m (2e-6 rad of carrier phase); gain product 3e-6 of the peak
// for analytic apertures (the kernel's cubic through four nodes is ~3e-8 away), 3e-5 with tabulated patterns (the
// bilinear table's kinks dominate).
constexpr long double kGuardPathTol = 2e-8L, kGuardGainTol = 3e-6L, kGuardGainTolLut = 3e-5L;
constexpr double kGuardMaxOffsetM = 4.0;         // |o_c| the fixed-point channel terms of K2k are scaled for
constexpr double kGuardMaxSlices = 30000.0;      // |path - window start| in range slices the 16.48 fixed point holds

// One velocity of the scene points (uniform current, or a corner of the current map's bounding box).
bool geometry_keyframes_ok_at(const sim_instrument *in, const sim_geometry *g, const sim_scene *sc, int H,
                              const long double vel[3])
{
    const int P = g->n_pulses, C = in->n_channels;
    const int n_keys = (P - 1 + H - 1) / H + 1;
    long double o_fd = 0;
    for (int c = 0; c < C; ++c) o_fd = std::max<long double>(o_fd, std::fabs(in->channel_offset_m[c]));
    // Tabulated patterns: the kernel's cubic through four lookups follows a bilinear table only as closely as the
    // table follows a smooth function; 2.63 = 1 + the Lebesgue constant 1.63 of the four-point cubic.  The lattice
    // check below samples the rest; together they must stay inside kGuardGainTolLut.
    const bool lut = in->tx_pattern || in->rx_pattern;
    long double kink = 0, gain_tol = kGuardGainTol;
    if (lut) {
        long double dt_, gt_, dr_, gr_;
        table_roughness(in, 0, dt_, gt_);
        table_roughness(in, 1, dr_, gr_);
        kink = 2.63L * (dt_ * gr_ + dr_ * gt_);
        gain_tol = kGuardGainTolLut;
        if (!(kink <= gain_tol)) return false;
    }
    // a direction that leaves a table's grid inside an interval sees the hard edge of reading G29 (zero gain outside):
    // no polynomial follows that step, so every sampled direction must stay one cell inside the grid
    auto inside = [&](int k, long double ua, long double ue) {
        const float *tab = k ? in->rx_pattern : in->tx_pattern;
        if (!tab) return true;
        const int nu = k ? in->rx_pattern_nu : in->tx_pattern_nu, nv = k ? in->rx_pattern_nv : in->tx_pattern_nv;
        const double *ur = k ? in->rx_pattern_u : in->tx_pattern_u, *vr = k ? in->rx_pattern_v : in->tx_pattern_v;
        const long double gu = (ua - ur[0]) * (nu - 1) / ((long double)ur[1] - ur[0]);
        const long double gv = (ue - vr[0]) * (nv - 1) / ((long double)vr[1] - vr[0]);
        return gu >= 1 && gu <= nu - 2 && gv >= 1 && gv <= nv - 2;
    };
    const long double fsc = (long double)in->fs_hz / kC0, half_len = 0.5L * in->chirp_len_s * in->fs_hz;
    for (int gx = -1; gx <= 1; ++gx)
        for (int gy = -1; gy <= 1; ++gy) {
            const long double x0 = sc->centre_m[0] + gx * 0.5L * (sc->nx - 1) * sc->spacing_m;
            const long double y0 = sc->centre_m[1] + gy * 0.5L * (sc->ny - 1) * sc->spacing_m;
            auto at = [&](int p, long double pos[3]) {
                pos[0] = x0 + vel[0] * g->t_pulse_s[p]; pos[1] = y0 + vel[1] * g->t_pulse_s[p]; pos[2] = sc->centre_m[2];
            };
            for (int j = 0; j + 1 < n_keys; ++j) {
                const int k0 = std::min(j * H, P - 1), k1 = std::min((j + 1) * H, P - 1);
                if (k1 <= k0) continue;
                long double pa[3], pb[3];
                at(k0, pa); at(k1, pb);
                const GuardEval e0 = guard_eval(in, g, k0, pa, vel, o_fd), e1 = guard_eval(in, g, k1, pb, vel, o_fd);
                const long double t0 = g->t_pulse_s[k0], h = (long double)g->t_pulse_s[k1] - t0;
                if (!(h > 0)) return false;
                if (lut && !(inside(0, e0.uat, e0.uet) && inside(1, e0.uar, e0.uer) && inside(1, e0.uao, e0.ueo) &&
                             inside(0, e1.uat, e1.uet) && inside(1, e1.uar, e1.uer) && inside(1, e1.uao, e1.ueo)))
                    return false;
                // the part of the channel path difference that is linear in t is rounded to an integer by one FP32 FMA: it
                // must stay under 2^21 units of 2^-32 range slice (and of `mult` 2^-32 turns, scaled inside the kernel)
                for (int c = 0; c < C; ++c)
                    if (!(fabsl(e1.dl[c] - e0.dl[c]) * fsc * 4294967296.0L < 2097152.0L)) return false;
                // the kernel's gain interpolant: cubic through s = 0, 1/3, 2/3, 1 with the direction cosines between
                // the keyframes interpolated linearly; channel term by one finite difference at mid-interval
                cld Pn[4];
                for (int n = 0; n < 4; ++n) {
                    const long double sn = n / 3.0L;
                    Pn[n] = host_gain(in, 0, e0.uat + sn * (e1.uat - e0.uat), e0.uet + sn * (e1.uet - e0.uet)) *
                            host_gain(in, 1, e0.uar + sn * (e1.uar - e0.uar), e0.uer + sn * (e1.uer - e0.uer));
                }
                const cld c1 = 0.5L * (-11.0L * Pn[0] + 18.0L * Pn[1] - 9.0L * Pn[2] + 2.0L * Pn[3]);
                const cld c2 = 4.5L * (2.0L * Pn[0] - 5.0L * Pn[1] + 4.0L * Pn[2] - Pn[3]);
                const cld c3 = 4.5L * (-Pn[0] + 3.0L * Pn[1] - 3.0L * Pn[2] + Pn[3]);
                const cld gtm = host_gain(in, 0, 0.5L * (e0.uat + e1.uat), 0.5L * (e0.uet + e1.uet));
                const cld grm = host_gain(in, 1, 0.5L * (e0.uar + e1.uar), 0.5L * (e0.uer + e1.uer));
                const cld gom = host_gain(in, 1, 0.5L * (e0.uao + e1.uao), 0.5L * (e0.ueo + e1.ueo));
                const cld bq = o_fd > 0 ? gtm * (gom - grm) / o_fd : cld(0, 0);
                for (int p = k0; p <= k1; ++p) {
                    long double pp[3];
                    at(p, pp);
                    const GuardEval ex = guard_eval(in, g, p, pp, vel, o_fd);
                    // the kernel steps the interval by pulse INDEX (uniform pulse times): a jittered PRF fails here
                    const long double s = (long double)(p - k0) / (long double)(k1 - k0), s2 = s * s, s3 = s2 * s;
                    const long double Rh = (2 * s3 - 3 * s2 + 1) * e0.R + (s3 - 2 * s2 + s) * h * e0.Rd +
                                           (-2 * s3 + 3 * s2) * e1.R + (s3 - s2) * h * e1.Rd;
                    if (!(fabsl(Rh - ex.R) <= kGuardPathTol)) return false;
                    // inside the range of the kernel's fixed point (and of its window arithmetic)
                    if (!(fabsl((ex.R - (long double)kC0 * g->t0_s[p]) * fsc - half_len) <= kGuardMaxSlices)) return false;
                    if (!(fabsl((long double)kC0 * ((long double)g->t0_s[p] - g->t0_s[k0]) * fsc) <= kGuardMaxSlices)) return false;
                    if (lut && !(inside(0, ex.uat, ex.uet) && inside(1, ex.uar, ex.uer) && inside(1, ex.uao, ex.ueo))) return false;
                    const cld Pq = Pn[0] + s * (c1 + s * (c2 + s * c3));
                    for (int c = 0; c < C; ++c) {
                        const long double dl = e0.dl[c] + s * (e1.dl[c] - e0.dl[c]);
                        if (!(fabsl(dl - ex.dl[c]) <= kGuardPathTol)) return false;
                        const cld gq = Pq + (long double)in->channel_offset_m[c] * bq;
                        if (!(std::abs(gq - ex.gtc * ex.grc[c]) + kink <= gain_tol)) return false;
                    }
                }
            }
        }
    return true;
}

bool geometry_keyframes_ok(const sim_instrument *in, const sim_geometry *g, const sim_scene *sc, int H,
                           const float cur_lo[2], const float cur_hi[2])
{
    const int P = g->n_pulses, C = in->n_channels;
    if (H <= 1 || H + 1 > kMaxKeyPulses || C > kMaxKeyChannels) return false;
    for (int c = 0; c < C; ++c) if (!(std::fabs(in->channel_offset_m[c]) <= kGuardMaxOffsetM)) return false;
    const double ratio = in->f0_hz / in->fs_hz;
    if (!(ratio > 0.0 && ratio < 65000.0)) return false;
    // uniform pulse times inside every interval (the waves are stepped by pulse index too; the platform terms are
    // checked against the exact geometry below)
    const int n_keys = (P - 1 + H - 1) / H + 1;
    for (int j = 0; j + 1 < n_keys; ++j) {
        const int k0 = std::min(j * H, P - 1), k1 = std::min((j + 1) * H, P - 1);
        if (k1 <= k0) continue;
        const double h = g->t_pulse_s[k1] - g->t_pulse_s[k0];
        for (int p = k0; p <= k1; ++p)
            if (!(std::fabs(g->t_pulse_s[p] - (g->t_pulse_s[k0] + h * (double)(p - k0) / (double)(k1 - k0))) <= 1e-9)) return false;
    }
    if (!sc->current_mps) {
        const long double vel[3] = {sc->current_uniform[0], sc->current_uniform[1], 0.0L};
        return geometry_keyframes_ok_at(in, g, sc, H, vel);
    }
    // a current map: the four corners of the bounding box of its values (the drift of a scene point enters the
    // interpolants through its velocity and its position at every pulse)
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
            const long double vel[3] = {a ? cur_hi[0] : cur_lo[0], b ? cur_hi[1] : cur_lo[1], 0.0L};
            if (!geometry_keyframes_ok_at(in, g, sc, H, vel)) return false;
        }
    return true;
}

}  // namespace

extern "C" {

const char *sim_error_string(int code)
{
    switch (code) {
        case SIM_OK: return "ok";
        case SIM_EINVAL: return "invalid argument";
        case SIM_ERANGE: return "pulse range out of bounds";
        case SIM_ENOMEM: return "out of memory";
        case SIM_ECUDA: return "CUDA error";
        default: return "unknown error";
    }
}

const char *sim_last_cuda_error(const sim_handle *h) { return h ? h->cuda_err.c_str() : ""; }

void sim_destroy(sim_handle *h)
{
    if (!h) return;
    DeviceGuard g(h->device);
    h->xt.release(); h->yt.release(); h->tt.release(); h->chirp_n.release(); h->carrier_p.release();
    h->wk.release(); h->carrier_frac.release(); h->pulses.release();
    h->sigma0.release(); h->current.release(); h->xi.release(); h->xi_polar.release();
    h->pattern[0].release(); h->pattern[1].release();
    h->xi_state.release(); h->beta_g.release(); h->doppler_turns.release(); h->xi_t.release();
    h->z.release(); h->slope.release(); h->slope_t.release(); h->dxy.release();
    h->zt.release(); h->zc.release(); h->ztc.release(); h->zttc.release(); h->slopec.release(); h->slope_tc.release(); h->dxy_t.release(); h->omega.release(); h->recs.release(); h->tinfo.release();
    h->tspan.release(); h->acc.release(); h->counters.release(); h->out_staging.release();
    h->mom.release(); h->cspec.release(); h->tw.release(); h->cspec2.release(); h->tw2.release(); h->band.release();
    delete h;
}

int sim_create(const sim_instrument *in, const sim_geometry *g, const sim_scene *sc, const sim_options *opts,
               int device, sim_handle **out)
{
    if (!out) return SIM_EINVAL;
    *out = nullptr;
    int rc = validate(in, g, sc);
    if (rc != SIM_OK) return rc;
    if (opts && opts->tile_facets != 0) {
        int t = opts->tile_facets;
        if (t < 4 || t > 64 || (t & (t - 1))) return SIM_EINVAL;
    }
    if (opts && (opts->accumulate_mode < 0 || opts->accumulate_mode > 2)) return SIM_EINVAL;
    if (opts && (opts->kinematics_keyframe < 0 || opts->kinematics_keyframe > 4096)) return SIM_EINVAL;
    if (opts && (opts->geometry_keyframe < 0 || opts->geometry_keyframe > 1)) return SIM_EINVAL;
    if (opts && opts->fft_band != 0 && opts->fft_band != 1) {
        const int n = opts->fft_band;
        if (n < 256 || n > 8192 || (n & (n - 1))) return SIM_EINVAL;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return SIM_ECUDA;
    }
    sim_handle *h = new (std::nothrow) sim_handle();
    if (!h) return SIM_ENOMEM;
    h->device = device;
    DeviceGuard guard(device);
    if (!guard.ok) { delete h; return SIM_ECUDA; }

    const int P = g->n_pulses, C = in->n_channels, Nw = sc->n_waves, nx = sc->nx, ny = sc->ny;
    const int Ns = in->n_samples;
    const double lambda = kC0 / in->f0_hz;
    DevParams &prm = h->prm;
    h->n_pulses = P;
    h->n_facets = (int64_t)nx * ny;
    h->chirp_rate = in->chirp_rate_hz_per_s; h->chirp_len = in->chirp_len_s; h->fs = in->fs_hz;
    prm.nx = nx; prm.ny = ny; prm.spacing = sc->spacing_m;
    prm.cx = sc->centre_m[0]; prm.cy = sc->centre_m[1]; prm.cz = sc->centre_m[2];
    prm.n_samples = Ns; prm.n_channels = C; prm.n_mid = Ns / 2;
    prm.inv_lambda = in->f0_hz / kC0;
    prm.fs_over_c0 = in->fs_hz / kC0;
    prm.kappa = in->chirp_rate_hz_per_s / (2.0 * in->fs_hz * in->fs_hz);
    prm.len = in->chirp_len_s * in->fs_hz;
    prm.half_len = 0.5 * prm.len;
    prm.ap_tx_a = in->tx_aperture_m[0] / lambda; prm.ap_tx_e = in->tx_aperture_m[1] / lambda;
    prm.ap_rx_a = in->rx_aperture_m[0] / lambda; prm.ap_rx_e = in->rx_aperture_m[1] / lambda;
    prm.cull_thr = (in->cull_two_way_db > -300.0) ? (float)std::pow(10.0, in->cull_two_way_db / 20.0) : 0.f;
    prm.n_waves = Nw; prm.choppy = sc->choppy ? 1 : 0; prm.tilt = sc->tilt_modulation ? 1 : 0;
    prm.has_sigma0 = sc->sigma0_lin ? 1 : 0; prm.has_current = sc->current_mps ? 1 : 0;
    prm.sigma0_uniform = sc->sigma0_uniform; prm.look_x = sc->look_dir[0]; prm.look_y = sc->look_dir[1];
    prm.cur_ux = sc->current_uniform[0]; prm.cur_uy = sc->current_uniform[1];
    h->need_slope = prm.tilt != 0;

    // ---- accumulation mode (SIM_ACCUMULATE_*): the spectral path needs an integer replica length
    //      (one waveform kernel for every facet) and a transform that fits shared memory ----
    const double len_round = std::nearbyint(prm.len);
    const bool len_integer = std::fabs(prm.len - len_round) < 1e-9 * std::max(1.0, prm.len) && len_round >= 1.0;
    int nfft = 256;
    while (nfft < Ns + (int)len_round - 1 && nfft < (1 << 20)) nfft <<= 1;
    bool spectral_ok = len_integer && nfft <= 16384;
    std::vector<std::complex<double>> ck_host;
    if (spectral_ok) {
        // truncation of the Chebyshev series at Kt moments: an under-sampled chirp (B > ~fs) needs more than Kt = 8
        std::vector<double> cmax;
        chebyshev_kernels(prm.kappa, (int)len_round, kMomentOrder + 4, ck_host, cmax);
        double tail = 0;
        for (int k = kMomentOrder; k < kMomentOrder + 4; ++k) tail += cmax[k];
        if (!(tail <= kMomentTruncationTol)) spectral_ok = false;
    }
    const int mode = opts ? opts->accumulate_mode : SIM_ACCUMULATE_AUTO;
    if (mode == SIM_ACCUMULATE_SPECTRAL && !spectral_ok) { delete h; return SIM_EINVAL; }
    h->spectral = (mode == SIM_ACCUMULATE_SPECTRAL) || (mode == SIM_ACCUMULATE_AUTO && spectral_ok);
    h->replica = (int)len_round;
    h->nfft = nfft;
    h->nb = Ns + h->replica - 1;
    h->nb_pad = (h->nb + 3) & ~3;

    // ---- tiling: a spatial tile must stay narrow in delay compared with the replica ----
    const double grad = std::max(0.25, path_gradient_l1(g, sc));
    const double samples_per_facet = sc->spacing_m * grad * prm.fs_over_c0;   // delay spread per facet step
    int tile = opts ? opts->tile_facets : 0;
    if (h->spectral) {
        if (tile == 0) tile = 32;
        tile = std::min(tile, 32);                                // facet state lives in registers (moments.cu)
    } else if (tile == 0) {
        tile = 64;
        const double budget = std::max(16.0, prm.len / 12.0);     // spread <= ~8 % of the replica
        while (tile > 8 && tile * samples_per_facet > budget) tile >>= 1;
    }
    prm.tile = tile;
    prm.tiles_x = (nx + tile - 1) / tile; prm.tiles_y = (ny + tile - 1) / tile;
    prm.n_tiles = prm.tiles_x * prm.tiles_y;
    prm.tile_cap = tile * tile;
    double wave_sum = 0;
    const WaveView wv = wave_view(sc);
    for (int n = 0; n < wv.n_nodes; ++n) {
        double a1 = 0;
        for (int w = 0; w < Nw; ++w) a1 += std::fabs(wv.amp[(size_t)n * Nw + w]);
        wave_sum = std::max(wave_sum, wv.hetero ? 2.0 * a1 : a1);
    }
    const double tile_spread = tile * samples_per_facet + 2.0 * 2.0 * wave_sum * prm.fs_over_c0 + 3.0;
    h->accum = accumulate_plan(prm, tile_spread);
    if (!h->spectral && h->accum.block_threads > 1024) { delete h; return SIM_EINVAL; }   // replica too long for one CTA of the direct form
    h->span_cap_m = std::min(4064, (((int)std::ceil(tile_spread) + 8) + 31) & ~31);
    {   // K2k's own tiling (sheared) and the slice window of its tiles
        // 32 x 32 tiles of the spectral path become 32 x 24 sheared tiles here: 256 threads x 3 facets, two CTAs per SM
        // (4 facets per thread spill, 2 leave the slices half as full: profiles/r2_k2k_history.md)
        const int k2k_cap = (prm.tile_cap == 1024) ? 768 : prm.tile_cap;
        const ShearPlan sp = plan_sheared_tiles(g, sc, prm.fs_over_c0, k2k_cap);
        prm.k2k_cap = k2k_cap;
        prm.k2k_w = sp.w; prm.k2k_h = sp.h; prm.k2k_axis = sp.axis; prm.k2k_a0 = sp.a0; prm.k2k_shear = sp.shear;
        prm.k2k_tiles_a = sp.tiles_a; prm.k2k_n_tiles = sp.tiles_a * sp.tiles_b;
        const double spread_k = sp.extent + 2.0 * 2.0 * wave_sum * prm.fs_over_c0 + 3.0;
        h->span_cap_k = std::min(4064, (((int)std::ceil(spread_k) + 8) + 15) & ~15);
    }

    {   // receive-channel legs by series (geometry_common.cuh): offsets small against the nearest range
        double o_max = 0, r_min = 1e300;
        for (int c = 0; c < C; ++c) o_max = std::max(o_max, std::fabs(in->channel_offset_m[c]));
        const double radius = 0.5 * std::hypot(nx * sc->spacing_m, ny * sc->spacing_m) + 4.0 * wave_sum + 100.0;
        for (int p = 0; p < P; ++p) {
            const double *r = g->rx_pos_m + 3 * p;
            const double d = std::sqrt((r[0] - sc->centre_m[0]) * (r[0] - sc->centre_m[0]) +
                                       (r[1] - sc->centre_m[1]) * (r[1] - sc->centre_m[1]) +
                                       (r[2] - sc->centre_m[2]) * (r[2] - sc->centre_m[2]));
            r_min = std::min(r_min, d - radius);
        }
        prm.series_channels = (r_min > 0 && o_max <= 1e-4 * r_min) ? 1 : 0;
    }
    h->key_H = choose_keyframe_spacing(g, sc, opts ? opts->kinematics_keyframe : 0);
    {   // K2k's fixed point: f0 / fs in 2^-48 units; the constant phase of the slice bias
        const long double ratio = (long double)in->f0_hz / (long double)in->fs_hz;
        if (ratio > 0 && ratio < 65000.0L) {
            const long double k48 = ratio * 281474976710656.0L;       // 2^48
            const unsigned long long K = (unsigned long long)(k48 + 0.5L);
            prm.ratio_hi = (uint32_t)(K >> 32); prm.ratio_lo = (uint32_t)K;
            // the kernel multiplies by K 2^-48, not by f0 / fs itself: the bias uses the same number
            const long double kr = (long double)K / 281474976710656.0L;
            long double turns = (32768.0L - 0.5L * (long double)prm.len) * kr;
            turns -= floorl(turns);
            prm.phase_bias32 = (uint32_t)(unsigned long long)(turns * 4294967296.0L + 0.5L);
        }
        if (sc->current_mps) {
            for (int k = 0; k < 2; ++k) { h->cur_lo[k] = 1e30f; h->cur_hi[k] = -1e30f; }
            const size_t n2 = 2 * (size_t)nx * ny;
            for (size_t k = 0; k < n2; ++k) {
                h->cur_lo[k & 1] = std::min(h->cur_lo[k & 1], sc->current_mps[k]);
                h->cur_hi[k & 1] = std::max(h->cur_hi[k & 1], sc->current_mps[k]);
            }
            for (int k = 0; k < 2; ++k) {                  // room for sim_update_scene
                const float m = 0.25f * std::max({std::fabs(h->cur_lo[k]), std::fabs(h->cur_hi[k]), 0.1f});
                h->cur_lo[k] -= m; h->cur_hi[k] += m;
            }
        }
    }
    prm.lut_any = (in->tx_pattern || in->rx_pattern) ? 1 : 0;
    if (h->spectral && h->key_H > 1 && prm.series_channels && C <= kMaxKeyChannels &&
        !(opts && opts->geometry_keyframe == 1)) {
        // keyframed geometry: the spacing the wave bound admits, halved until the geometry bounds hold too
        // (a forced spacing is tried as it is)
        const bool forced = opts && opts->kinematics_keyframe > 1;
        for (int H = h->key_H; H > 1; H = forced ? 1 : H / 2) {
            if (H + 1 <= kMaxKeyPulses && moments_keyframed_fits(prm, h->span_cap_k) &&
                geometry_keyframes_ok(in, g, sc, H, h->cur_lo, h->cur_hi)) {
                h->key_H = H; h->geo_keyframed = true;
                break;
            }
        }
    }
    if (h->geo_keyframed && !prm.choppy && !(opts && opts->kinematics_keyframe > 1))
        h->key_H1 = choose_coarse_spacing(g, sc, h->key_H);
    // ---- batch size ----
    const int64_t fcap = (int64_t)prm.n_tiles * prm.tile_cap;
    const int64_t surf_row = h->n_facets * 8 + (h->need_slope ? h->n_facets * 8 : 0) +
                             (prm.choppy ? h->n_facets * 16 : 0);
    const int64_t per_pulse_common = h->key_H > 1 ? 2 * surf_row / h->key_H + 1 : surf_row;
    h->speckle_ar1 = sc->speckle_tau_s > 0;
    h->nodes_x = sc->wave_nodes_x > 0 ? sc->wave_nodes_x : 0; h->nodes_y = h->nodes_x ? sc->wave_nodes_y : 0;
    h->node_spacing = sc->wave_node_spacing_m;
    h->seed = sc->seed;
    const int64_t per_pulse = per_pulse_common + (h->speckle_ar1 ? h->n_facets * 8 : 0) +
        (h->spectral ? (int64_t)C * kMomentOrder * h->nb_pad * 8
                     : (int64_t)C * fcap * (int64_t)sizeof(Rec) + (int64_t)C * Ns * 16 +
                           (int64_t)prm.n_tiles * (4 + 16 * C));
    // default workspace: 16 GiB, at most a quarter of the free device memory, at least 1 GiB (a small cap splits a dwell
    // of a large scene into many batches, and every batch recomputes the keyframe rows at its ends: on 2^26 facets
    // a 4 GiB cap made three batches of 64 pulses and K1 computed 12 rows instead of 5)
    int64_t ws = (opts && opts->workspace_bytes > 0) ? opts->workspace_bytes : ((int64_t)16 << 30);
    if (!(opts && opts->workspace_bytes > 0)) {
        size_t mem_free = 0, mem_total = 0;
        if (cudaMemGetInfo(&mem_free, &mem_total) == cudaSuccess)
            ws = std::max<int64_t>((int64_t)1 << 30, std::min<int64_t>(ws, (int64_t)(mem_free / 4)));
        else cudaGetLastError();
    }
    int pb = (int)std::max<int64_t>(1, std::min<int64_t>(ws / std::max<int64_t>(per_pulse, 1), h->spectral ? 1024 : 256));
    if (opts && opts->pulses_per_batch > 0) pb = opts->pulses_per_batch;
    pb = std::min(pb, P);
    if (!(opts && opts->pulses_per_batch > 0)) {        // balance the batches of a full-dwell call
        const int pb_max = pb;
        const int nb = (P + pb - 1) / pb;
        pb = (P + nb - 1) / nb;
        // Decoupled keyframes: every batch evaluates the coarse rows (spacing H1) that span it, four rows per thread block
        // of K1 (three where that wastes none; a partial group costs a whole one), so batch boundaries on coarse keyframes
        // save rows: Large, 2048 pulses, at most 900 per batch: 3 x 683 pulses = 3 x 7 rows = 24 row slots; 896 + 896 + 256
        // = 8 + 8 + 3 rows = 19.
        if (h->key_H1 > 0 && pb < P) {
            auto row_slots = [&](int batch) {
                int slots = 0;
                for (int p0 = 0; p0 < P; p0 += batch) {
                    int first = 0, rows = 0;
                    surface_rows(h, p0, std::min(batch, P - p0), &first, &rows, h->key_H1);
                    slots += kinematics_coarse_row_slots(rows);
                }
                return slots;
            };
            int best = pb, best_slots = row_slots(pb);
            for (int cand = h->key_H1; cand <= pb_max; cand += h->key_H1) {
                const int sl = row_slots(cand);
                if (sl < best_slots || (sl == best_slots && cand > best)) { best = cand; best_slots = sl; }
            }
            pb = best;
        }
    }
    h->pulses_per_batch = pb;

    // ---- host tables (fp64) ----
    // one set per node of the heterogeneous lattice (a single set on the homogeneous surface); row q = node * Nw + w
    const size_t NQ = (size_t)wv.n_nodes * Nw;
    std::vector<double2> xt(NQ * nx), yt(NQ * ny), tt(NQ * P);
    std::vector<float4> wk(NQ);
    for (size_t q = 0; q < NQ; ++q) {
        const double kx = wv.kx[q], ky = wv.ky[q], amp = wv.amp[q], om = wv.omega[q], ph = wv.phase[q];
        for (int i = 0; i < nx; ++i) {
            double x = sc->centre_m[0] + (i - 0.5 * (nx - 1)) * sc->spacing_m;
            double a = kx * x;
            xt[q * nx + i] = make_double2(amp * std::cos(a), amp * std::sin(a));
        }
        for (int j = 0; j < ny; ++j) {
            double y = sc->centre_m[1] + (j - 0.5 * (ny - 1)) * sc->spacing_m;
            double a = ky * y + ph;
            yt[q * ny + j] = make_double2(std::cos(a), std::sin(a));
        }
        for (int p = 0; p < P; ++p) {
            double a = -om * g->t_pulse_s[p];
            tt[q * P + p] = make_double2(std::cos(a), std::sin(a));
        }
        double k = std::hypot(kx, ky);
        wk[q] = make_float4((float)kx, (float)ky, k > 0 ? (float)(kx / k) : 0.f, k > 0 ? (float)(ky / k) : 0.f);
    }
    std::vector<PulseConst> pcs(P);
    std::vector<double2> carrier(P);
    std::vector<double> cfrac(P);
    for (int p = 0; p < P; ++p) {
        PulseConst &pc = pcs[p];
        std::memset(&pc, 0, sizeof(pc));
        pc.t = g->t_pulse_s[p];
        pc.r0 = kC0 * g->t0_s[p];
        const double *v = g->rx_vel_mps + 3 * p;
        const double vn = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        for (int k = 0; k < 3; ++k) {
            pc.tx_pos[k] = g->tx_pos_m[3 * p + k];
            pc.tx_a[k] = g->tx_frame[9 * p + 3 + k]; pc.tx_e[k] = g->tx_frame[9 * p + 6 + k];
            pc.rx_a[k] = g->rx_frame[9 * p + 3 + k]; pc.rx_e[k] = g->rx_frame[9 * p + 6 + k];
            pc.rx_ref[k] = g->rx_pos_m[3 * p + k];
            for (int c = 0; c < C; ++c) pc.rx_pos[c][k] = g->rx_pos_m[3 * p + k] + in->channel_offset_m[c] * v[k] / vn;
            pc.rx_vhat[k] = v[k] / vn;
            pc.tx_vel[k] = g->tx_vel_mps[3 * p + k]; pc.rx_vel[k] = v[k];
            pc.rx_va += pc.rx_vhat[k] * pc.rx_a[k];
            pc.rx_ve += pc.rx_vhat[k] * pc.rx_e[k];
        }
        for (int c = 0; c < C; ++c) pc.ch_off[c] = in->channel_offset_m[c];
        // carrier phase of the reference path: f0 * (r0/c0), reduced in long double
        long double cyc = (long double)pc.r0 * ((long double)in->f0_hz / (long double)kC0);
        long double fr = cyc - floorl(cyc);
        cfrac[p] = (double)fr;
        carrier[p] = make_double2(std::cos(-2.0 * M_PI * (double)fr), std::sin(-2.0 * M_PI * (double)fr));
    }
    std::vector<double2> chirp(Ns);
    for (int n = 0; n < Ns; ++n) {
        long double m = (long double)(n - prm.n_mid);
        long double turns = (long double)prm.kappa * m * m;
        turns -= floorl(turns);
        chirp[n] = make_double2(std::cos(2.0 * M_PI * (double)turns), std::sin(2.0 * M_PI * (double)turns));
    }

    // ---- device allocation + upload ----
    auto bail = [&](int code) { sim_destroy(h); return code; };
#define CKC(call)                                                                 \
    do {                                                                          \
        cudaError_t e__ = (call);                                                 \
        if (e__ != cudaSuccess) { int c__ = fail_cuda(h, e__, #call); return bail(c__); } \
    } while (0)
    CKC(h->xt.alloc(xt.size())); CKC(h->yt.alloc(yt.size())); CKC(h->tt.alloc(tt.size()));
    CKC(h->wk.alloc(wk.size())); CKC(h->pulses.alloc(P)); CKC(h->carrier_p.alloc(P));
    CKC(h->carrier_frac.alloc(P)); CKC(h->chirp_n.alloc(Ns));
    if (Nw) {
        CKC(cudaMemcpy(h->xt.p, xt.data(), xt.size() * sizeof(double2), cudaMemcpyHostToDevice));
        CKC(cudaMemcpy(h->yt.p, yt.data(), yt.size() * sizeof(double2), cudaMemcpyHostToDevice));
        CKC(cudaMemcpy(h->tt.p, tt.data(), tt.size() * sizeof(double2), cudaMemcpyHostToDevice));
        CKC(cudaMemcpy(h->wk.p, wk.data(), wk.size() * sizeof(float4), cudaMemcpyHostToDevice));
    }
    CKC(cudaMemcpy(h->pulses.p, pcs.data(), (size_t)P * sizeof(PulseConst), cudaMemcpyHostToDevice));
    CKC(cudaMemcpy(h->carrier_p.p, carrier.data(), (size_t)P * sizeof(double2), cudaMemcpyHostToDevice));
    CKC(cudaMemcpy(h->carrier_frac.p, cfrac.data(), (size_t)P * sizeof(double), cudaMemcpyHostToDevice));
    CKC(cudaMemcpy(h->chirp_n.p, chirp.data(), (size_t)Ns * sizeof(double2), cudaMemcpyHostToDevice));
    const size_t F = (size_t)h->n_facets;
    if (sc->sigma0_lin) {
        CKC(h->sigma0.alloc(F));
        CKC(cudaMemcpy(h->sigma0.p, sc->sigma0_lin, F * sizeof(float), cudaMemcpyHostToDevice));
    }
    if (sc->current_mps) {
        CKC(h->current.alloc(F));
        CKC(cudaMemcpy(h->current.p, sc->current_mps, F * sizeof(float2), cudaMemcpyHostToDevice));
    }
    {
        const float *tab[2] = {in->tx_pattern, in->rx_pattern};
        const int32_t nu[2] = {in->tx_pattern_nu, in->rx_pattern_nu}, nv[2] = {in->tx_pattern_nv, in->rx_pattern_nv};
        const double *ur[2] = {in->tx_pattern_u, in->rx_pattern_u}, *vr[2] = {in->tx_pattern_v, in->rx_pattern_v};
        for (int k = 0; k < 2; ++k) {
            PatternLut &L = prm.lut[k];
            L = PatternLut{};
            if (!tab[k]) continue;
            const size_t n = (size_t)nu[k] * nv[k];
            CKC(h->pattern[k].alloc(n));
            CKC(cudaMemcpy(h->pattern[k].p, tab[k], n * sizeof(float2), cudaMemcpyHostToDevice));
            L.tab = h->pattern[k].p; L.nu = nu[k]; L.nv = nv[k];
            L.u0 = ur[k][0]; L.su = (nu[k] - 1) / (ur[k][1] - ur[k][0]);
            L.v0 = vr[k][0]; L.sv = (nv[k] - 1) / (vr[k][1] - vr[k][0]);
        }
    }
    CKC(h->xi.alloc(F));
    if (sc->xi) {
        CKC(cudaMemcpy(h->xi.p, sc->xi, F * sizeof(float2), cudaMemcpyHostToDevice));
    } else {
        CKC(launch_speckle_from_seed(h->xi.p, (int64_t)F, sc->seed, nullptr));
    }
    CKC(h->xi_polar.alloc(F));
    CKC(launch_speckle_polar(h->xi.p, h->xi_polar.p, (int64_t)F, nullptr));
    if (h->speckle_ar1) {
        std::vector<float2> bg(P);
        std::vector<uint32_t> dop(P);
        for (int p = 0; p < P; ++p) {
            const double beta = p ? std::exp(-(g->t_pulse_s[p] - g->t_pulse_s[p - 1]) / sc->speckle_tau_s) : 1.0;
            bg[p] = make_float2((float)beta, (float)std::sqrt(std::max(0.0, 1.0 - beta * beta)));
            const long double turns = (long double)sc->speckle_doppler_hz * (long double)g->t_pulse_s[p];
            const long double fr = turns - floorl(turns);
            dop[p] = (uint32_t)(unsigned long long)(fr * 4294967296.0L + 0.5L);
        }
        CKC(h->beta_g.alloc(P)); CKC(h->doppler_turns.alloc(P)); CKC(h->xi_state.alloc(F));
        CKC(h->xi_t.alloc(F * (size_t)pb));
        CKC(cudaMemcpy(h->beta_g.p, bg.data(), (size_t)P * sizeof(float2), cudaMemcpyHostToDevice));
        CKC(cudaMemcpy(h->doppler_turns.p, dop.data(), (size_t)P * sizeof(uint32_t), cudaMemcpyHostToDevice));
    }
    CKC(cudaDeviceSynchronize());
    {
        const size_t rows = h->key_H > 1 ? (size_t)(pb / h->key_H + 3) : (size_t)pb;
        h->surf_rows_cap = (int)rows;
        CKC(h->z.alloc(F * rows));
        if (h->need_slope) CKC(h->slope.alloc(F * rows));
        if (prm.choppy) CKC(h->dxy.alloc(F * rows));
        if (h->key_H > 1) {
            CKC(h->zt.alloc(F * rows));
            if (prm.choppy) CKC(h->dxy_t.alloc(F * rows));
        }
        if (h->key_H1 > 0) {
            const size_t rows1 = (size_t)(pb / h->key_H1 + 3);
            CKC(h->zc.alloc(F * rows1)); CKC(h->ztc.alloc(F * rows1)); CKC(h->zttc.alloc(F * rows1));
            if (h->need_slope) { CKC(h->slopec.alloc(F * rows1)); CKC(h->slope_tc.alloc(F * rows1)); }
        }
        CKC(h->omega.alloc(std::max<size_t>(NQ, 1)));
        if (NQ) CKC(cudaMemcpy(h->omega.p, wv.omega, NQ * sizeof(double), cudaMemcpyHostToDevice));
    }
    if (!h->spectral) {
        CKC(h->recs.alloc((size_t)C * pb * fcap));
        CKC(h->tinfo.alloc((size_t)pb * prm.n_tiles));
        CKC(h->tspan.alloc((size_t)C * pb * prm.n_tiles));
        CKC(h->acc.alloc((size_t)C * pb * Ns));
    } else {
        // waveform kernels c_k[m] (chebyshev_kernels above), their spectra, and the transform's twiddle table
        const int L = h->replica;
        std::vector<float2> ck((size_t)kMomentOrder * L), tw((size_t)nfft);
        for (int k = 0; k < kMomentOrder; ++k)
            for (int m = 0; m < L; ++m) {
                const std::complex<double> v = ck_host[(size_t)k * L + m];
                ck[(size_t)k * L + m] = make_float2((float)v.real(), (float)v.imag());
            }
        for (int k = 0; k < nfft; ++k) {
            const double a = -2.0 * M_PI * (double)k / (double)nfft;
            tw[k] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
        DevBuf<float2> d_ck;
        CKC(d_ck.alloc(ck.size()));
        CKC(h->tw.alloc(tw.size()));
        CKC(h->cspec.alloc((size_t)kMomentOrder * nfft));
        CKC(cudaMemcpy(d_ck.p, ck.data(), ck.size() * sizeof(float2), cudaMemcpyHostToDevice));
        CKC(cudaMemcpy(h->tw.p, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice));
        cudaError_t e_spec = launch_kernel_spectra(nfft, d_ck.p, L, h->tw.p, h->cspec.p, nullptr);
        if (e_spec == cudaSuccess) e_spec = cudaDeviceSynchronize();
        // band transform (fftconv.cu): K2k records the slice range every vector occupies; size from the scene's extent
        // in slices -- only an estimate, a vector with a wider band takes the full transform
        h->nfft2 = 0;
        const int band_opt = opts ? opts->fft_band : 0;
        if (e_spec == cudaSuccess && h->geo_keyframed && band_opt != 1) {
            int n2 = 256;
            if (band_opt > 1) n2 = band_opt;
            else {
                const double need = scene_slice_extent(in, g, sc, wave_sum) * prm.fs_over_c0 + 16.0 + (L - 1);
                while (n2 < need && n2 < nfft) n2 <<= 1;
            }
            if (n2 < nfft && n2 >= L) {                  // else: no smaller transform holds a band plus the replica
                std::vector<float2> tw2((size_t)n2);
                for (int k = 0; k < n2; ++k) {
                    const double a = -2.0 * M_PI * (double)k / (double)n2;
                    tw2[k] = make_float2((float)std::cos(a), (float)std::sin(a));
                }
                e_spec = h->tw2.alloc(tw2.size());
                if (e_spec == cudaSuccess) e_spec = h->cspec2.alloc((size_t)kMomentOrder * n2);
                if (e_spec == cudaSuccess) e_spec = h->band.alloc((size_t)2 * C * pb);
                if (e_spec == cudaSuccess) e_spec = cudaMemcpy(h->tw2.p, tw2.data(), tw2.size() * sizeof(float2), cudaMemcpyHostToDevice);
                if (e_spec == cudaSuccess) e_spec = launch_kernel_spectra(n2, d_ck.p, L, h->tw2.p, h->cspec2.p, nullptr);
                if (e_spec == cudaSuccess) e_spec = cudaDeviceSynchronize();
                if (e_spec == cudaSuccess) h->nfft2 = n2;
            }
        }
        d_ck.release();
        CKC(e_spec);
        CKC(h->mom.alloc((size_t)C * pb * kMomentOrder * h->nb_pad));
    }
    CKC(h->counters.alloc(2));
    CKC(cudaMemset(h->counters.p, 0, 2 * sizeof(unsigned long long)));
#undef CKC
    h->stats.tile_facets = tile; h->stats.pulses_per_batch = pb; h->stats.n_tiles = prm.n_tiles;
    h->stats.accumulate_block_threads = h->accum.block_threads;
    h->stats.accumulate_mode = h->spectral ? SIM_ACCUMULATE_SPECTRAL : SIM_ACCUMULATE_DIRECT;
    h->stats.fft_size = h->spectral ? nfft : 0;
    h->stats.kinematics_keyframe = h->key_H;
    h->stats.geometry_keyframed = h->geo_keyframed ? 1 : 0;
    h->stats.fft_band_size = h->spectral ? h->nfft2 : 0;
    h->stats.kinematics_coarse_keyframe = (h->geo_keyframed && h->key_H1 > 0) ? h->key_H1 : 0;
    *out = h;
    return SIM_OK;
}

// `host_dst` non-null: `out` is the device staging buffer and every finished batch is copied to
// host_dst (same [C][n_out][Ns] layout) on the handle's copy stream while the next batch computes.
static int run_batches(sim_handle *h, int32_t pb0, int32_t pb1, float2 *out, cudaStream_t s,
                       int batch_pulses = 0, float2 *host_dst = nullptr)
{
    const DevParams &prm = h->prm;
    const int n_out = pb1 - pb0;
    const int batch = batch_pulses > 0 ? std::min(batch_pulses, h->pulses_per_batch) : h->pulses_per_batch;
    int64_t launches = 0;
    size_t copies = 0;
    auto ship = [&](int p0, int n_pl) -> cudaError_t {
        if (!host_dst) return cudaSuccess;
        if (copies == h->copy_events.size()) {
            cudaEvent_t e;
            cudaError_t rc = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
            if (rc != cudaSuccess) return rc;
            h->copy_events.push_back(e);
        }
        cudaEvent_t e = h->copy_events[copies++];
        cudaError_t rc = cudaEventRecord(e, s);
        if (rc == cudaSuccess) rc = cudaStreamWaitEvent(h->copy_stream, e, 0);
        const size_t row = (size_t)prm.n_samples * sizeof(float2);
        const size_t off = (size_t)(p0 - pb0) * prm.n_samples;
        if (rc == cudaSuccess)
            rc = cudaMemcpy2DAsync(host_dst + off, (size_t)n_out * row, out + off, (size_t)n_out * row,
                                   (size_t)n_pl * row, prm.n_channels, cudaMemcpyDeviceToHost, h->copy_stream);
        return rc;
    };
    CK(h, cudaMemsetAsync(h->counters.p, 0, 2 * sizeof(unsigned long long), s));
    h->events_used = 0;
    auto mark = [&]() -> cudaError_t {
        if (!h->profiling) return cudaSuccess;
        if (h->events_used == h->events.size()) {
            cudaEvent_t e;
            cudaError_t rc = cudaEventCreate(&e);
            if (rc != cudaSuccess) return rc;
            h->events.push_back(e);
        }
        return cudaEventRecord(h->events[h->events_used++], s);
    };
    const SurfBufs bufs{h->z.p, h->zt.p, h->slope.p, h->slope_t.p, h->dxy.p, h->dxy_t.p};
    for (int p0 = pb0; h->spectral && p0 < pb1; p0 += batch) {
        const int n_pl = std::min(batch, pb1 - p0);
        // the moment rows are zeroed on a second stream, beside K1 (which does not touch them): forked after whatever
        // precedes on `s` (the previous batch's K3s reads the rows), joined before K2k
        if (!h->aux_stream) {
            CK(h, cudaStreamCreateWithFlags(&h->aux_stream, cudaStreamNonBlocking));
            CK(h, cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
            CK(h, cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
        }
        CK(h, cudaEventRecord(h->ev_fork, s));
        CK(h, cudaStreamWaitEvent(h->aux_stream, h->ev_fork, 0));
        CK(h, cudaMemsetAsync(h->mom.p, 0, (size_t)prm.n_channels * n_pl * kMomentOrder * h->nb_pad * sizeof(float2), h->aux_stream));
        CK(h, cudaEventRecord(h->ev_join, h->aux_stream));
        CK(h, mark());
        MomentArgs ma{};
        { int rc = run_kinematics(h, bufs, p0, n_pl, s, &ma.surf, h->geo_keyframed && h->key_H1 > 0); if (rc != SIM_OK) return rc; }
        CK(h, mark());
        ma.pulses = h->pulses.p;
        ma.sigma0 = h->sigma0.p; ma.current = h->current.p;
        { int rc = run_speckle(h, p0, n_pl, s, &ma.xi_polar, &ma.xi_pulse_stride); if (rc != SIM_OK) return rc; }
        ma.mom = h->mom.p; ma.nb_pad = h->nb_pad; ma.replica = h->replica;
        ma.span_cap = h->geo_keyframed ? h->span_cap_k : h->span_cap_m;
        ma.dbg_slice = h->dbg_slice; ma.dbg_eps = h->dbg_eps; ma.dbg_w = h->dbg_w; ma.dbg_keep = h->dbg_keep; ma.dbg_pulse = h->dbg_pulse;
        ma.counters = h->counters.p;
        const size_t n_vec = (size_t)prm.n_channels * n_pl;
        if (h->nfft2) {                                  // lo preset to 0x7f7f7f7f, hi to 0x80808080
            ma.band_lo = h->band.p; ma.band_hi = h->band.p + n_vec;
            CK(h, cudaMemsetAsync(ma.band_lo, 0x7f, n_vec * sizeof(int32_t), s));
            CK(h, cudaMemsetAsync(ma.band_hi, 0x80, n_vec * sizeof(int32_t), s));
        }
        CK(h, cudaStreamWaitEvent(s, h->ev_join, 0));
        if (h->geo_keyframed) CK(h, launch_moments_keyframed(prm, ma, p0, n_pl, s));
        else CK(h, launch_moments(prm, ma, p0, n_pl, s));
        CK(h, mark());
        FftConvArgs fa{};
        fa.mom = h->mom.p; fa.cspec = h->cspec.p; fa.tw = h->tw.p; fa.carrier_p = h->carrier_p.p;
        fa.out = out; fa.n_out_pulses = n_out; fa.out_pulse0 = p0 - pb0;
        fa.nfft = h->nfft; fa.nb = h->nb; fa.nb_pad = h->nb_pad; fa.replica = h->replica;
        if (h->nfft2) {
            fa.band_lo = ma.band_lo; fa.band_hi = ma.band_hi; fa.cspec2 = h->cspec2.p; fa.tw2 = h->tw2.p; fa.nfft2 = h->nfft2;
        }
        CK(h, launch_fftconv(prm, fa, p0, n_pl, s));
        CK(h, mark());
        CK(h, mark());                                   // K4 slot: finalize is fused into K3s
        CK(h, ship(p0, n_pl));
        launches += 3 + (h->speckle_ar1 ? 1 : 0) + (h->nfft2 ? 1 : 0) + ((h->geo_keyframed && h->key_H1 > 0) ? 1 : 0);
    }
    for (int p0 = pb0; !h->spectral && p0 < pb1; p0 += batch) {
        const int n_pl = std::min(batch, pb1 - p0);
        CK(h, cudaMemsetAsync(h->acc.p, 0, (size_t)prm.n_channels * n_pl * prm.n_samples * sizeof(double2), s));
        CK(h, mark());
        GeometryArgs ga{};
        { int rc = run_kinematics(h, bufs, p0, n_pl, s, &ga.surf); if (rc != SIM_OK) return rc; }
        CK(h, mark());
        ga.pulses = h->pulses.p;
        ga.sigma0 = h->sigma0.p; ga.current = h->current.p; ga.xi = h->xi.p;
        { int rc = run_speckle(h, p0, n_pl, s, &ga.xi_polar, &ga.xi_pulse_stride); if (rc != SIM_OK) return rc; }
        ga.recs = h->recs.p; ga.tinfo = h->tinfo.p; ga.tspan = h->tspan.p; ga.counters = h->counters.p;
        ga.carrier_frac_t0 = h->carrier_frac.p;
        CK(h, launch_geometry(prm, ga, p0, n_pl, s));
        CK(h, mark());
        AccumulateArgs aa{h->recs.p, h->tinfo.p, h->tspan.p, h->acc.p, h->accum.block_threads,
                          h->accum.samples_per_thread, h->accum.warps_per_span, h->accum.span_cap, h->accum.smem_bytes};
        CK(h, launch_accumulate(prm, aa, n_pl, s));
        CK(h, mark());
        FinalizeArgs fa{h->acc.p, h->chirp_n.p, h->carrier_p.p, out, n_out, p0 - pb0};
        CK(h, launch_finalize(prm, fa, p0, n_pl, s));
        CK(h, mark());
        CK(h, ship(p0, n_pl));
        launches += 4 + (h->speckle_ar1 ? 1 : 0);
    }
    h->stats.kernel_launches = launches;
    h->stats.facet_echoes_nominal = h->n_facets * (int64_t)n_out * prm.n_channels;
    return SIM_OK;
}

int sim_generate(sim_handle *h, int32_t pulse_begin, int32_t pulse_end, void *iq_dev, void *cuda_stream)
{
    if (!h) return SIM_EINVAL;
    if (pulse_begin < 0 || pulse_end > h->n_pulses || pulse_begin >= pulse_end) return SIM_ERANGE;
    if (!iq_dev) return SIM_EINVAL;
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    return run_batches(h, pulse_begin, pulse_end, static_cast<float2 *>(iq_dev), static_cast<cudaStream_t>(cuda_stream));
}

int sim_generate_host(sim_handle *h, int32_t pulse_begin, int32_t pulse_end, void *iq_host, void *cuda_stream)
{
    if (!h) return SIM_EINVAL;
    if (pulse_begin < 0 || pulse_end > h->n_pulses || pulse_begin >= pulse_end) return SIM_ERANGE;
    if (!iq_host) return SIM_EINVAL;
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t n = (size_t)h->prm.n_channels * (pulse_end - pulse_begin) * h->prm.n_samples;
    {   // page-locked, device-accessible host memory (cudaHostAlloc / cudaHostRegister under unified addressing): the
        // last kernel of every batch stores the IQ samples straight into it -- the transfer over PCIe runs inside
        // that kernel instead of after it, no staging buffer, no copy
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, iq_host) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer) {
            int rc = run_batches(h, pulse_begin, pulse_end, static_cast<float2 *>(at.devicePointer), s);
            if (rc != SIM_OK) return rc;
            CK(h, cudaStreamSynchronize(s));
            return SIM_OK;
        }
        (void)cudaGetLastError();                        // pageable memory: not an error, staged below
    }
    if (h->out_staging.n < n) CK(h, h->out_staging.alloc(n));
    if (!h->copy_stream) CK(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
    // the workspace-sized batches of the call are shipped as they finish (splitting a dwell that fits one batch
    // costs more in K1 / K2k efficiency than the overlapped copy returns: measured on ATI)
    int rc = run_batches(h, pulse_begin, pulse_end, h->out_staging.p, s, 0, static_cast<float2 *>(iq_host));
    if (rc != SIM_OK) return rc;
    CK(h, cudaStreamSynchronize(h->copy_stream));
    CK(h, cudaStreamSynchronize(s));
    return SIM_OK;
}

int sim_update_scene(sim_handle *h, const float *sigma0_lin, const float *current_mps, const float *xi, void *cuda_stream)
{
    if (!h) return SIM_EINVAL;
    if ((sigma0_lin && !h->sigma0.p) || (current_mps && !h->current.p)) return SIM_EINVAL;
    {
        const size_t Fn = (size_t)h->n_facets;
        if (sigma0_lin) {
            const float lo[2] = {0.f, 0.f}, hi[2] = {3.4e38f, 3.4e38f};
            if (!floats_ok(sigma0_lin, Fn, lo, hi)) return SIM_EINVAL;
        }
        // the keyframed geometry was admitted for the current extremes seen at sim_create
        if (current_mps && !floats_ok(current_mps, 2 * Fn, h->cur_lo, h->cur_hi)) return SIM_EINVAL;
        if (xi && !finite_all(xi, 2 * Fn)) return SIM_EINVAL;
    }
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t F = (size_t)h->n_facets;
    if (sigma0_lin) CK(h, cudaMemcpyAsync(h->sigma0.p, sigma0_lin, F * sizeof(float), cudaMemcpyHostToDevice, s));
    if (current_mps) CK(h, cudaMemcpyAsync(h->current.p, current_mps, F * sizeof(float2), cudaMemcpyHostToDevice, s));
    if (xi) {
        CK(h, cudaMemcpyAsync(h->xi.p, xi, F * sizeof(float2), cudaMemcpyHostToDevice, s));
        CK(h, launch_speckle_polar(h->xi.p, h->xi_polar.p, (int64_t)F, s));
        h->xi_state_pulse = -1;                          // the cached AR(1) state started from the old xi
    }
    return SIM_OK;
}

int sim_replica(const sim_handle *h, float *host_c64_out, int32_t *n)
{
    if (!h || !n) return SIM_EINVAL;
    // samples m with -T/2 <= m/fs - T/2 < T/2  <=>  0 <= m < T fs
    const int32_t L = (int32_t)std::ceil(h->chirp_len * h->fs - 1e-9);
    *n = L;
    if (!host_c64_out) return SIM_OK;
    for (int32_t m = 0; m < L; ++m) {
        const double u = m / h->fs - 0.5 * h->chirp_len;
        const double ph = M_PI * h->chirp_rate * u * u;
        host_c64_out[2 * m] = (float)std::cos(ph);
        host_c64_out[2 * m + 1] = (float)std::sin(ph);
    }
    return SIM_OK;
}

int sim_debug_facets(sim_handle *h, int32_t pulse, double *pos, double *slope, double *tau, double *g_tx,
                     double *g_rx, double *amp, int32_t *keep)
{
    if (!h) return SIM_EINVAL;
    if (pulse < 0 || pulse >= h->n_pulses) return SIM_ERANGE;
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    const DevParams &prm = h->prm;
    const size_t F = (size_t)h->n_facets, C = prm.n_channels;
    DevBuf<double> d_pos, d_tau, d_gtx, d_grx, d_amp;
    DevBuf<int32_t> d_keep;
    DevBuf<float2> d_slope, d_slope_out;
    DevBuf<Rec> d_recs;                  // spectral handles own no record workspace
    DevBuf<TileInfo> d_tinfo;
    DevBuf<TileSpan> d_tspan;
    int rc = SIM_OK;
    auto run = [&]() -> int {
        Rec *recs = h->recs.p; TileInfo *tinfo = h->tinfo.p; TileSpan *tspan = h->tspan.p;
        if (!recs) {
            CK(h, d_recs.alloc(C * (size_t)prm.n_tiles * prm.tile_cap)); CK(h, d_tinfo.alloc(prm.n_tiles));
            CK(h, d_tspan.alloc(C * (size_t)prm.n_tiles));
            recs = d_recs.p; tinfo = d_tinfo.p; tspan = d_tspan.p;
        }
        CK(h, d_pos.alloc(3 * F)); CK(h, d_tau.alloc(C * F)); CK(h, d_gtx.alloc(F));
        CK(h, d_grx.alloc(C * F)); CK(h, d_amp.alloc(2 * C * F)); CK(h, d_keep.alloc(F));
        // the slope is reported even when the scene does not use it: temporary rows
        SurfBufs bufs{h->z.p, h->zt.p, h->slope.p, h->slope_t.p, h->dxy.p, h->dxy_t.p};
        if (!bufs.slope) {
            CK(h, d_slope.alloc(F * 3 * 2));
            bufs.slope = d_slope.p;
        }
        GeometryArgs ga{};
        { int rc2 = run_kinematics(h, bufs, pulse, 1, nullptr, &ga.surf); if (rc2 != SIM_OK) return rc2; }
        ga.pulses = h->pulses.p;
        // per-facet slope of this pulse (interpolated like K2 sees it), for the report only
        CK(h, d_slope_out.alloc(F));
        CK(h, launch_surface_slope(prm, ga.surf, h->pulses.p, pulse, d_slope_out.p, nullptr));
        if (!h->need_slope) ga.surf.slope = nullptr;
        ga.sigma0 = h->sigma0.p; ga.current = h->current.p; ga.xi = h->xi.p;
        { int rc2 = run_speckle(h, pulse, 1, nullptr, &ga.xi_polar, &ga.xi_pulse_stride); if (rc2 != SIM_OK) return rc2; }
        ga.recs = recs; ga.tinfo = tinfo; ga.tspan = tspan; ga.counters = nullptr;
        ga.dbg_pos = d_pos.p; ga.dbg_tau = d_tau.p; ga.dbg_gtx = d_gtx.p; ga.dbg_grx = d_grx.p;
        ga.dbg_amp = d_amp.p; ga.dbg_keep = d_keep.p; ga.carrier_frac_t0 = h->carrier_frac.p;
        CK(h, launch_geometry(prm, ga, pulse, 1, nullptr));
        CK(h, cudaDeviceSynchronize());
        if (pos) CK(h, cudaMemcpy(pos, d_pos.p, 3 * F * sizeof(double), cudaMemcpyDeviceToHost));
        if (tau) CK(h, cudaMemcpy(tau, d_tau.p, C * F * sizeof(double), cudaMemcpyDeviceToHost));
        if (g_tx) CK(h, cudaMemcpy(g_tx, d_gtx.p, F * sizeof(double), cudaMemcpyDeviceToHost));
        if (g_rx) CK(h, cudaMemcpy(g_rx, d_grx.p, C * F * sizeof(double), cudaMemcpyDeviceToHost));
        if (amp) CK(h, cudaMemcpy(amp, d_amp.p, 2 * C * F * sizeof(double), cudaMemcpyDeviceToHost));
        if (keep) CK(h, cudaMemcpy(keep, d_keep.p, F * sizeof(int32_t), cudaMemcpyDeviceToHost));
        if (slope) {
            std::vector<float2> tmp(F);
            CK(h, cudaMemcpy(tmp.data(), d_slope_out.p, F * sizeof(float2), cudaMemcpyDeviceToHost));
            for (size_t f = 0; f < F; ++f) { slope[2 * f] = tmp[f].x; slope[2 * f + 1] = tmp[f].y; }
        }
        return SIM_OK;
    };
    rc = run();
    h->xi_state_pulse = -1;                              // the debug pass walked the AR(1) speckle state: the next batch replays it
    d_pos.release(); d_tau.release(); d_gtx.release(); d_grx.release(); d_amp.release(); d_keep.release();
    d_slope.release(); d_slope_out.release(); d_recs.release(); d_tinfo.release(); d_tspan.release();
    return rc;
}

int sim_debug_echoes(sim_handle *h, int32_t pulse, int32_t *slice, float *eps, float *weight, int32_t *keep,
                     int64_t *n_edge_ambiguous)
{
    if (!h) return SIM_EINVAL;
    if (pulse < 0 || pulse >= h->n_pulses) return SIM_ERANGE;
    if (!h->spectral || !h->geo_keyframed || h->prm.lut_any || h->speckle_ar1) return SIM_EINVAL;
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    const size_t F = (size_t)h->n_facets, C = h->prm.n_channels;
    DevBuf<int32_t> d_slice, d_keep;
    DevBuf<float> d_eps;
    DevBuf<float2> d_w, d_out;
    auto run = [&]() -> int {
        CK(h, d_slice.alloc(C * F)); CK(h, d_keep.alloc(F)); CK(h, d_eps.alloc(C * F)); CK(h, d_w.alloc(C * F));
        CK(h, d_out.alloc(C * (size_t)h->prm.n_samples));
        CK(h, cudaMemset(d_slice.p, 0, C * F * sizeof(int32_t))); CK(h, cudaMemset(d_keep.p, 0, F * sizeof(int32_t)));
        CK(h, cudaMemset(d_eps.p, 0, C * F * sizeof(float))); CK(h, cudaMemset(d_w.p, 0, C * F * sizeof(float2)));
        h->dbg_slice = d_slice.p; h->dbg_keep = d_keep.p; h->dbg_eps = d_eps.p; h->dbg_w = d_w.p; h->dbg_pulse = pulse;
        const sim_stats saved = h->stats;
        const int rc = run_batches(h, pulse, pulse + 1, d_out.p, nullptr);
        h->stats = saved;
        h->dbg_slice = h->dbg_keep = nullptr; h->dbg_eps = nullptr; h->dbg_w = nullptr; h->dbg_pulse = -1;
        if (rc != SIM_OK) return rc;
        CK(h, cudaDeviceSynchronize());
        std::vector<int32_t> hk(F);
        std::vector<float> he(C * F);
        CK(h, cudaMemcpy(hk.data(), d_keep.p, F * sizeof(int32_t), cudaMemcpyDeviceToHost));
        CK(h, cudaMemcpy(he.data(), d_eps.p, C * F * sizeof(float), cudaMemcpyDeviceToHost));
        if (slice) CK(h, cudaMemcpy(slice, d_slice.p, C * F * sizeof(int32_t), cudaMemcpyDeviceToHost));
        if (weight) CK(h, cudaMemcpy(weight, d_w.p, C * F * sizeof(float2), cudaMemcpyDeviceToHost));
        if (eps) std::memcpy(eps, he.data(), C * F * sizeof(float));
        if (keep) std::memcpy(keep, hk.data(), F * sizeof(int32_t));
        if (n_edge_ambiguous) {
            int64_t n = 0;
            for (size_t c = 0; c < C; ++c)
                for (size_t f = 0; f < F; ++f)
                    if (hk[f] && (he[c * F + f] < 1e-6f || he[c * F + f] > 1.f - 1e-6f)) ++n;
            *n_edge_ambiguous = n;
        }
        return SIM_OK;
    };
    const int rc = run();
    h->xi_state_pulse = -1;                              // (the debug pass walked the speckle state)
    d_slice.release(); d_keep.release(); d_eps.release(); d_w.release(); d_out.release();
    return rc;
}

int sim_get_stats(sim_handle *h, sim_stats *out)
{
    if (!h || !out) return SIM_EINVAL;
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    unsigned long long c[2] = {0, 0};
    CK(h, cudaMemcpy(c, h->counters.p, sizeof(c), cudaMemcpyDeviceToHost));   // synchronises with prior work
    h->stats.facet_echoes_kept = (int64_t)c[0];
    h->stats.facet_samples = (int64_t)c[1];
    *out = h->stats;
    return SIM_OK;
}

int sim_set_profiling(sim_handle *h, int32_t enable)
{
    if (!h) return SIM_EINVAL;
    h->profiling = enable != 0;
    return SIM_OK;
}

int sim_get_kernel_ms(sim_handle *h, float ms[4])
{
    if (!h || !ms) return SIM_EINVAL;
    DeviceGuard g(h->device);
    if (!g.ok) return SIM_ECUDA;
    for (int k = 0; k < 4; ++k) ms[k] = 0.f;
    if (h->events_used == 0) return SIM_OK;
    CK(h, cudaEventSynchronize(h->events[h->events_used - 1]));
    for (size_t b = 0; b + 5 <= h->events_used; b += 5) {
        for (int k = 0; k < 4; ++k) {
            float t = 0.f;
            CK(h, cudaEventElapsedTime(&t, h->events[b + k], h->events[b + k + 1]));
            ms[k] += t;
        }
    }
    return SIM_OK;
}

}  // extern "C"
