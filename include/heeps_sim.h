/*
 * heeps_sim.h -- C ABI of the B200-native HEEPS/MARE raw-data generator hot path.
 *
 * The library computes, for every pulse p and receive phase-centre channel c, the complex
 * IQ samples
 *
 *   s_{c,p}[n] = sum_f a_f G_tx G_rx exp(-j 2 pi f0 tau_f)
 *                      rect((t_n - tau_f)/T) exp(j pi K (t_n - tau_f)^2),  t_n = t0[p] + n/fs
 *
 * (BASELINE.json north_star; scalar form of PAPER.md eq. (3) line 91 and eq. (16);
 * the range-slice sum of eq. (17), with the waveform convolution written
 * out).  Every step runs in hand-written CUDA kernels for sm_100a:
 *   K1 facet kinematics            (PAPER.md:53-55   surface = sum of wave components)
 *   K2 geometry + gains + amplitude + cull + tile bucketing
 *                                  (PAPER.md:91-98 ranges/phase, :202 antenna patterns, :223 contributing subset)
 *   K3 echo accumulation
 *   K4 finalize                    (raw data output)
 *
 * Conventions
 *   - All descriptor arrays are HOST pointers, C order, copied during sim_create (the caller
 *     may free them after it returns).  Units: SI (m, s, Hz, m/s); sigma0 linear (not dB).
 *   - Frame arrays are [P][3][3] with rows {boresight, azimuth axis, elevation axis}, unit,
 *     mutually orthogonal (checked to 1e-6).
 *   - Facet (i,j), i fastest, rest position centre + ((i-(nx-1)/2) d, (j-(ny-1)/2) d, 0).
 *   - Output is complex64 [C][pulse_end-pulse_begin][Ns], interleaved (re,im) float32.
 *   - Return value 0 on success, a negative SIM_E* code otherwise.  Nothing is printed, no
 *     exception or abort crosses the boundary.  A handle is not thread-safe and serves ONE stream at
 *     a time (its workspace and its cached speckle state are shared by its calls); distinct handles are independent.  There is no CPU fallback: without a CUDA device every
 *     compute entry point returns SIM_ECUDA.
 *   - Echo samples falling outside [0, Ns) are clipped silently (not an error).
 */
#ifndef HEEPS_SIM_H
#define HEEPS_SIM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SIM_OK        0
#define SIM_EINVAL   (-1)   /* null pointer, bad size, NaN (descriptors and per-facet maps), non-orthonormal frame, > SIM_MAX_CHANNELS */
#define SIM_ERANGE   (-2)   /* pulse range outside [0, P] or empty-inverted */
#define SIM_ENOMEM   (-3)   /* host or device allocation failed */
#define SIM_ECUDA    (-4)   /* CUDA runtime error; see sim_last_cuda_error */

#define SIM_MAX_CHANNELS 8

typedef struct sim_handle sim_handle;        /* opaque, owned by the library */

/* Instrument (BASELINE.json north_star (d): carrier, chirp rate/length, fs, PRF, apertures, offsets) */
typedef struct {
    double f0_hz;                  /* carrier */
    double chirp_rate_hz_per_s;    /* K = B/T, > 0 up-chirp; p(t) = rect(t/T) exp(j pi K t^2)  (reading G2) */
    double chirp_len_s;            /* T */
    double fs_hz;                  /* complex sampling rate */
    double prf_hz;                 /* informational; pulse times come from sim_geometry */
    int32_t n_samples;             /* Ns fast-time samples per pulse */
    double tx_aperture_m[2];       /* {azimuth length, elevation height}; field pattern sinc*sinc (G5); 0 = isotropic */
    double rx_aperture_m[2];
    int32_t n_channels;            /* C, 1..SIM_MAX_CHANNELS */
    const double *channel_offset_m;/* [C] host; along-track offsets about the Rx state vector (G8) */
    double cull_two_way_db;        /* facet dropped for all channels iff 20log10|G_t G_r,ref| < this; <= -300 disables (G6) */
    /* Antenna patterns as complex u-v grids.  A non-NULL table replaces that
     * antenna's analytic aperture pattern: complex field gain (re, im interleaved) on pattern_nv x pattern_nu nodes,
     * u = direction cosine along the azimuth axis over [pattern_u[0], pattern_u[1]] (first and last node), v likewise
     * along the elevation axis; bilinear between nodes, zero outside the grid (reading G29).  Time dependence (TOPSAR
     * steering) enters through the per-pulse frames of sim_geometry.  The keyframed geometry (sim_options.geometry_keyframe)
     * accepts a table only when it is fine enough for its three-point gain interpolant (node-to-node second differences
     * <= ~1e-4, checked at sim_create); a coarser table is looked up at every pulse. */
    const float *tx_pattern, *rx_pattern;              /* host [nv][nu][2] or NULL */
    int32_t tx_pattern_nu, tx_pattern_nv, rx_pattern_nu, rx_pattern_nv;
    double tx_pattern_u[2], tx_pattern_v[2], rx_pattern_u[2], rx_pattern_v[2];
} sim_instrument;

/* Geometry: per-pulse Tx/Rx state vectors (stop-and-go, reading G9) */
typedef struct {
    int32_t n_pulses;              /* P */
    const double *t_pulse_s;       /* [P] time at which the scene is frozen for pulse p */
    const double *tx_pos_m, *tx_vel_mps, *rx_pos_m, *rx_vel_mps;   /* [P][3] each */
    const double *tx_frame, *rx_frame;                             /* [P][3][3] */
    const double *t0_s;            /* [P] time of sample 0 after the Tx chirp centre (G1) */
} sim_geometry;

/* Scene: facet grid, wave components, sigma0 / current / speckle fields */
typedef struct {
    int32_t nx, ny;
    double spacing_m;              /* d; facet area A = d^2 (G15) */
    double centre_m[3];
    int32_t n_waves;               /* Nw >= 0 */
    const double *kx, *ky, *amp, *omega, *phase;   /* [Nw] host; z = sum A cos(kx x + ky y - omega t + phase) */
    int32_t choppy;                /* 0 linear surface; 1 Choppy Wave Model horizontal displacement */
    const float *sigma0_lin;       /* [ny][nx] host or NULL -> sigma0_uniform */
    double sigma0_uniform;
    int32_t tilt_modulation;       /* sigma0 *= max(0, 1 + 2 grad z . look_dir)  (G12) */
    double look_dir[2];            /* horizontal unit vector radar -> scene */
    const float *current_mps;      /* [ny][nx][2] host or NULL -> current_uniform; applied by advection (G10) */
    double current_uniform[2];
    const float *xi;               /* [ny][nx][2] host complex speckle, or NULL -> derived from seed (G14) */
    uint64_t seed;
    /* Time-dependent intra-facet speckle.  speckle_tau_s > 0: the speckle of
     * facet f at pulse p is s_f(t_p) = [R + i I](t_p) exp(2 i pi f_s t_p) (eq. 7) with the order-1 autoregressive model of
     * eq. (10), R(t + dt) = beta R(t) + sqrt(1 - beta^2) R', beta = exp(-dt/tau_s), stepped pulse by pulse from xi_f at
     * pulse 0; the innovations R' + i I' (variance 1/2 per part) come from Philox4x32-10 keyed by `seed`, counter
     * (f lo, f hi, pulse, 1), Box-Muller (reading G27).  speckle_tau_s <= 0 (default): xi_f constant over the dwell. */
    double speckle_tau_s;
    double speckle_doppler_hz;     /* f_s of eq. (7) */
    /* Heterogeneous surface.  wave_nodes_x > 0: kx..phase above are ignored; node
     * (a, b) of a lattice of step wave_node_spacing_m (the tile size L), node (0, 0) at the rest position of facet (0, 0),
     * carries its own table of n_waves components -- the homogeneous tile T2L centred on it.  The surface displacement,
     * slope and velocity at a rest point are those of the four corner tiles of its lattice cell blended with the
     * weights of eq. (2), W^i = sqrt((1 - |x^i - x|/L)(1 - |y^i - y|/L)) (eq. (1); reading G28).  The lattice must cover
     * the grid: (nx-1) d <= (wave_nodes_x-1) L, likewise in y; at least 2 x 2 nodes. */
    int32_t wave_nodes_x, wave_nodes_y;
    double wave_node_spacing_m;
    const double *node_kx, *node_ky, *node_amp, *node_omega, *node_phase;   /* [nodes_y][nodes_x][n_waves] host */
} sim_scene;

/* Echo accumulation.  Both evaluate the same defined sum:
 *   DIRECT   every facet-echo's chirp replica is generated and added sample by sample;
 *   SPECTRAL facet-echoes are summed into range slices (eq. 17) as Kt = 8 Chebyshev moments of the
 *            sub-slice position, and the slices are convolved with the waveform by FFT (the paper's
 *            "impulse response ... subsequently convolved by the waveform", with the sub-slice term
 *            kept to ~1e-6).  Needs T*fs integer, Ns + T*fs - 1 <= 16384 and a chirp that Kt = 8 moments resolve
 *            (Chebyshev tail <= 5e-6: B <~ fs).
 *   AUTO     SPECTRAL where it applies, DIRECT otherwise. */
#define SIM_ACCUMULATE_AUTO     0
#define SIM_ACCUMULATE_DIRECT   1
#define SIM_ACCUMULATE_SPECTRAL 2

/* Tunables; zero-initialise for defaults. */
typedef struct {
    int32_t tile_facets;           /* spatial tile side in facets (4..64, power of 2; SPECTRAL clamps to 32); 0 = auto */
    int32_t pulses_per_batch;      /* 0 = auto from workspace_bytes (balanced over the dwell; with decoupled keyframes the batch
                                      boundaries are put on coarse keyframes where that saves keyframe rows) */
    int64_t workspace_bytes;       /* cap for per-batch device workspace; 0 = 16 GiB, at most a quarter of the free device memory */
    int32_t accumulate_mode;       /* SIM_ACCUMULATE_*; SPECTRAL where it does not apply -> SIM_EINVAL */
    int32_t kinematics_keyframe;   /* wave sums evaluated exactly every H-th pulse (with time derivatives) and
                                      cubic-Hermite interpolated between: 0 = auto (largest H <= 64 whose error
                                      bound sum_w A_w (omega_w h)^4/384 <= 4e-8 m; slopes linear between, their error <= 1.2e-4), 1 = every pulse, n = force H = n.
                                      With the keyframed geometry (below), a linear surface and H chosen automatically the wave sums themselves
                                      are evaluated only every 4 H-th (or 2 H-th) pulse, with second time derivatives, and the rows at spacing H
                                      are their quintic (slopes: cubic) Hermite interpolants (bounds 1e-8 m, 1e-5) */
    int32_t geometry_keyframe;     /* SPECTRAL only: 0 = auto -- where kinematics keyframes are in use (H > 1), C <= 4, the
                                      receive offsets are small (|o_c| <= 4 m) and the pulse times inside every keyframe
                                      interval are uniform, ranges / gains are evaluated exactly at the keyframe pulses only
                                      and interpolated between (Hermite path length stepped by fixed-point forward differences,
                                      cubic gains), after sim_create has verified the interpolants against the exact geometry
                                      at every pulse on a lattice of scene points (path 2e-8 m, gains 3e-6; tabulated patterns:
                                      3e-5, and every sampled direction at least one cell inside the tables);
                                      1 = off (exact geometry at every pulse) */
    int32_t fft_band;              /* SPECTRAL with keyframed geometry: a vector whose echoes occupy a narrow band of range
                                      slices is convolved by a transform of that band alone: 0 = auto (size from the scene's
                                      slice extent), 1 = off (always the full Ns + L - 1 transform), n >= 256 (power of 2,
                                      < the full size) = that band transform; wider vectors always take the full one */
    int32_t reserved[4];
} sim_options;

/*
 * sim_create: validate descriptors, upload tables, allocate the per-batch workspace on CUDA
 * device `device`.  *out receives the handle.  opts may be NULL.
 */
int sim_create(const sim_instrument *inst, const sim_geometry *geo, const sim_scene *scene,
               const sim_options *opts, int device, sim_handle **out);

/*
 * sim_generate: IQ for pulses [pulse_begin, pulse_end) into caller-owned DEVICE memory
 * iq_dev (complex64 [C][pulse_end-pulse_begin][Ns]); asynchronous on cuda_stream (a
 * cudaStream_t, NULL = default stream); overwrites, never accumulates into, iq_dev;
 * idempotent per pulse range (that is the restart story).
 */
int sim_generate(sim_handle *h, int32_t pulse_begin, int32_t pulse_end, void *iq_dev, void *cuda_stream);

/*
 * sim_generate_host: same, but iq_host is HOST memory, and the call returns after the samples
 * are there (cuda_stream synchronised).  Page-locked memory the device can address
 * (cudaHostAlloc, cudaHostRegister, a pinned torch tensor) is written directly by the last
 * kernel of every batch: the PCIe transfer runs inside that kernel, nothing is staged or
 * copied.  Pageable memory goes through a device staging buffer, finished batches copied on
 * a second stream while the next batch computes.  Used for the end-to-end measurement.
 */
int sim_generate_host(sim_handle *h, int32_t pulse_begin, int32_t pulse_end, void *iq_host, void *cuda_stream);

/*
 * sim_update_scene: replace the per-facet maps from HOST arrays (any may be NULL = keep):
 * sigma0 [ny][nx], current [ny][nx][2], xi [ny][nx][2]; host->device copies on cuda_stream.
 * A map that was NULL (uniform) at sim_create cannot be introduced later (SIM_EINVAL).  The new maps are scanned
 * like the ones given to sim_create: finite, sigma0 >= 0, and every current component inside the range of the map
 * given at sim_create widened by a quarter (the keyframe guard was run for that range), else SIM_EINVAL.
 */
int sim_update_scene(sim_handle *h, const float *sigma0_lin, const float *current_mps, const float *xi,
                     void *cuda_stream);

/* sim_replica: the transmitted waveform samples exp(j pi K (m/fs - T/2)^2), m = 0..*n-1 (PAPER.md:209:
 * "raw data are output together with the waveforms").  host_c64_out may be NULL to query *n. */
int sim_replica(const sim_handle *h, float *host_c64_out, int32_t *n);

/* Per-facet intermediates of one pulse for unit parity (host arrays, any may be NULL):
 * pos [F][3], slope [F][2], tau [C][F], g_tx [F], g_rx [C][F], amp [C][F][2] (= a G_t G_r exp(-j2pi f0 tau)),
 * keep [F] (int32).  Synchronous. */
int sim_debug_facets(sim_handle *h, int32_t pulse, double *pos, double *slope, double *tau, double *g_tx,
                     double *g_rx, double *amp, int32_t *keep);

/* Per-facet-echo intermediates of the DEFAULT spectral path with keyframed geometry (moments_keyframed.cu), for one
 * pulse (host arrays, any may be NULL): range slice b = ceil((tau - t0) fs - T fs / 2) (the first in-window sample of
 * the echo; eq. (17): slice membership is an integer decision) slice [C][F]; sub-slice position
 * eps = b - ((tau - t0) fs - T fs / 2) in (0, 1], eps [C][F]; complex weight a G_t G_r,c exp(-j 2 pi f0 (tau - t0[p]))
 * as the kernel interpolates it, weight [C][F][2]; keep [F].  *n_edge_ambiguous = kept facet-echoes whose
 * position lies within 1e-6 of an integer: their slice may legitimately differ from an fp64 evaluation's (reading
 * G18).  SIM_EINVAL unless the handle runs the spectral form with keyframed geometry (sim_stats), analytic antenna
 * patterns and static speckle.  Synchronous. */
int sim_debug_echoes(sim_handle *h, int32_t pulse, int32_t *slice, float *eps, float *weight, int32_t *keep,
                     int64_t *n_edge_ambiguous);

/* Counters of the most recent sim_generate* call (after the stream has completed). */
typedef struct {
    int64_t facet_echoes_nominal;  /* F * pulses * C                                   */
    int64_t facet_echoes_kept;     /* after the cull                                   */
    int64_t facet_samples;         /* sum over kept facet-echoes of in-window samples (0 on the SPECTRAL path with keyframed geometry) */
    int64_t kernel_launches;       /* kernels launched by the call                     */
    int32_t tile_facets, pulses_per_batch, n_tiles, accumulate_block_threads;
    int32_t max_span_samples;      /* largest per-tile sample span seen                */
    int32_t accumulate_mode;       /* SIM_ACCUMULATE_DIRECT or _SPECTRAL, as resolved at sim_create */
    int32_t fft_size;              /* SPECTRAL: transform length; else 0              */
    int32_t kinematics_keyframe;   /* H as resolved at sim_create                     */
    int32_t geometry_keyframed;    /* 1 when ranges / gains are interpolated between keyframes (sim_options) */
    int32_t fft_band_size;         /* SPECTRAL: band transform length (sim_options.fft_band), 0 = not in use */
    int32_t kinematics_coarse_keyframe;   /* spacing at which the wave sums themselves are evaluated when it is a multiple of
                                             kinematics_keyframe (decoupled keyframes, sim_options.kinematics_keyframe); else 0 */
} sim_stats;
int sim_get_stats(sim_handle *h, sim_stats *out);

/* Per-kernel device time of the most recent call, measured with CUDA events on the caller's
 * stream when enabled (adds event records only): ms[0..3] = K1, K2, K3, K4 totals (SPECTRAL: K1 kinematics,
 * K2s geometry + moments, K3s FFT convolution + finalize, 0). */
int sim_set_profiling(sim_handle *h, int32_t enable);
int sim_get_kernel_ms(sim_handle *h, float ms[4]);

/* DIAGNOSTIC, not part of the method's boundary: pipe-throughput microbenchmarks on `device` (the FP32 / XU / FP64 pipe peaks that
 * bound the ALU-bound kernels are measured in the same run as the numbers quoted against them).
 * All figures are LANE operations per second at the clock the GPU ran the probe at (an FMA = 1
 * operation; a packed f32x2 instruction = 2).  Synchronous; takes a few tens of milliseconds. */
typedef struct {
    double ffma_per_s;            /* scalar FFMA                                      */
    double fadd_per_s;            /* scalar FADD                                      */
    double ffma2_lane_per_s;      /* packed FFMA2 (f32x2)                             */
    double fadd2_lane_per_s;      /* packed FADD2 (f32x2)                             */
    double mix_f32x2_lane_per_s;  /* FFMA2 and FADD2 alternating (the K3 inner loop)  */
    double mufu_per_s;            /* MUFU.SIN / MUFU.COS                              */
    double dfma_per_s;            /* DFMA                                             */
    int32_t sm_count;
    int32_t reserved[3];
} sim_pipe_peaks;
int sim_measure_pipe_peaks(int device, sim_pipe_peaks *out);

/*
 * sim_echoes_to_iq_static: the entry point that ALLOCATES NOTHING -- for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it).  It is the echo accumulation of the SPECTRAL form
 * (eq. (17) + waveform convolution; SIM_ACCUMULATE_SPECTRAL above) for ONE (channel, pulse) vector
 * from a caller-supplied list of facet-echoes:
 *
 *     iq[n] = phase * sum_e weight_e exp(j pi K ((n - slice_e + eps_e)/fs - T/2)^2)   over slice_e <= n < slice_e + T fs,
 *
 * i.e. echo e lays its chirp replica down from sample slice_e on, its delay ending eps_e in [0, 1] samples before that
 * sample (slice, eps, weight: what sim_debug_echoes reports).  No handle: the range-slice moment rows that the normal
 * path keeps in its cudaMalloc'd workspace, the waveform taps, their spectra and the FFT twiddles live in ONE static
 * device array inside the library (1.38 MB, held by every GPU that loads the library until exit), and the FFT
 * convolution kernel is the normal path's, launched on that array.  The call enqueues one memset and four kernels on
 * cuda_stream and returns; it calls no cudaMalloc, cudaFree or allocating library routine (first use on a device looks
 * the array's address up once, cudaGetSymbolAddress).
 *   slice_dev [n] int32, eps_dev [n] float, weight_dev [n][2] float (re, im): DEVICE memory, read only; n_echoes >= 0
 *   (0: the vector is zero-filled, the pointers may be NULL).  phase: HOST, {re, im} of the factor applied to the vector
 *   (the normal path's exp(-j 2 pi f0 t0[p])).  iq_dev: DEVICE complex64 [n_samples], overwritten.  Echoes whose window
 *   misses [0, n_samples) are clipped silently.
 * Limits: T fs an integer <= SIM_STATIC_MAX_REPLICA and n_samples + T fs - 1 <= SIM_STATIC_MAX_SLICES, else SIM_ERANGE
 * (nothing is launched); a chirp that eight moments do not resolve (B >~ fs), a non-integer T fs or bad arguments:
 * SIM_EINVAL; SIM_ECUDA on a CUDA error.
 * Every call uses the same array, which keeps the last call's contents (the call clears the rows it needs first):
 * calls that overlap on one GPU -- two streams, two threads, two captured graphs replayed concurrently -- RACE.  Serialise them.
 */
#define SIM_STATIC_MAX_SLICES  8192
#define SIM_STATIC_MAX_REPLICA 4096
int sim_echoes_to_iq_static(double chirp_rate_hz_per_s, double chirp_len_s, double fs_hz, int32_t n_samples,
                            const int32_t *slice_dev, const float *eps_dev, const float *weight_dev, int64_t n_echoes,
                            const double phase[2], void *iq_dev, int device, void *cuda_stream);

void sim_destroy(sim_handle *h);
const char *sim_error_string(int code);
/* Text of the last CUDA error seen by this handle ("" if none). Valid until the next call on h. */
const char *sim_last_cuda_error(const sim_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* HEEPS_SIM_H */
