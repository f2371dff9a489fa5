// K2k -- geometry, gains, amplitude, cull and range-slice moments with the GEOMETRY evaluated exactly only
// at the kinematics keyframes (SURVEY.md §8(a) A2..A6 moment form).
//
// moments.cu evaluates the fp64 antenna legs and the sinc patterns of every facet at every pulse: 1156
// instructions per facet-pulse, issue-bound (profiles/r1_v4).  But over one keyframe interval (H pulses, a few
// milliseconds) everything a facet-echo needs is a smooth function of time:
//
//   R(t)   = r_t + r_r,ref  bistatic path to the un-offset phase centre: cubic HERMITE from the exact values and
//            time derivatives at the two keyframes,  dR/dt = u_t.(v_f - V_tx) + u_r.(v_f - V_rx)  with the facet
//            velocity v_f = (current + dD_h/dt, dz/dt) from K1's rate rows.  Error <= h^4 max|d4R/dt4| / 384:
//            platform term 3 V^4/r^3 ~ 0.02 m/s^4 -> 4e-13 m at h = 9.4 ms; wave term = K1's own bound.
//   d_c(t) = r_r,c - r_r,ref  (receive phase centre c, |o_c| <= 16 m) = o_c a(t) + o_c^2 b, a = -(d.v^)/r linear
//            in t, b = (1 - a^2)/(2 r).
//   P(t)   = G_t G_r,ref      CUBIC through t0, t0 + h/3, t0 + 2h/3, t1 with the sinc arguments (direction cosines)
//            between the keyframes interpolated linearly (they are linear in t to ~1e-7): interpolation error ~3e-8
//            of the peak gain, so that the cull decision |P| >= threshold (G6) differs from the exact one only for
//            facets within ~1e-7 of the threshold (a quadratic left 4e-6: a handful of flipped facets per pulse on
//            the Large scene, each worth 2e-5 of relative L2).  G_r,c = G_r,ref + o_c dG/do with dG/do by one finite
//            difference at mid-interval.  |a_f|(t) (tilt modulation) quadratic through t0, t_mid, t1.
//
// sim_create verifies these interpolants against the exact geometry on a lattice of scene points at EVERY pulse
// (host, long double) and falls back to moments.cu when any bound fails (sim_api.cu geometry_keyframes_ok):
// non-smooth state vectors or non-uniform pulse times never reach this kernel.
//
// ARITHMETIC OF THE PULSE LOOP.  Pulse times inside an interval are uniform (checked on the host), so the cubic R is
// advanced from pulse to pulse by FORWARD DIFFERENCES in 64-bit fixed point: rho = (R - R_base) fs/c0 - L/2 + 2^15 in
// units of 2^-48 range slice (R_base = c0 t0 of the first keyframe, a CTA constant): three 64-bit adds per facet and
// pulse, no fp64 in the loop (the fp64 chain, its conversions and the per-echo sub-slice phase were two thirds of
// round 1's 100 instructions per facet-echo in this stage).  From the same word come
//   the slice and the sub-slice position  (rho - w_p + channel term) >> 16 = [integer slice . 32-bit fraction]
//       (w_p = the sampling window's own start (r0[p] - R_base) fs/c0: an arbitrary per-pulse input, from shared memory),
//   the carrier phase  -R/lambda = -rho (f0/fs) + const: the 32 fraction bits of the 64 x 64-bit product with f0/fs in
//       2^-48 units -- two IMAD.HI and one IMAD -- exact to 3 units of 2^-32 turn at any range.
// The receive-channel path difference o_c a(t) + o_c^2 b enters both words, and to the same accuracy (a facet-echo whose
// slice position sits within the error of an integer lands in the neighbouring slice, and since the replica's window
// is a hard edge every such echo costs two samples of its full amplitude: relative L2 sqrt(4 delta / L) for an error of
// delta slices at ANY scene size -- 1e-5 slices: 1.8e-4; 1e-8: 6e-6): a is split into its value at the tile centre (one
// exact word per channel and CTA, shared memory) and the facet's small deviation + its drift over the interval, which
// one FP32 FMA against 1.5 x 2^23 rounds to an integer.
// The chirp's own sub-slice phase kappa eps^2 is part of the waveform kernels (sim_api.cu builds them as the Chebyshev
// coefficients of the exact slice response), so the per-echo phase is the carrier phase alone.
//
// One CTA = one SHEARED spatial tile x one keyframe interval (256 threads x 3 facets -- 32 x 24 -- two CTAs per SM).  A thread holds
// its facets' interpolants in registers and loops over the interval's pulses.  The tile's facet-echoes (all C channels)
// are ordered by range slice ONCE per interval -- counting sort at its middle pulse: shared-memory histogram by integer
// ATOMS, scan, slot = first position of the slice + rank -- because over a few milliseconds a facet changes slice only
// when its sub-slice position crosses 0 or 1 (a percent or two of the echoes per pulse).  Per pulse: (A) slice,
// sub-slice position and complex weight of every facet-echo, branch-free; an echo found in its sorted slice writes its
// weight into its slot, one found elsewhere ("stray") leaves a zero there and goes to a short shared-memory list; one
// barrier; (C) 8 threads per occupied slice (one work list over all channels) sum the Kt Chebyshev moments of the
// slice's contiguous slots (packed FFMA2), transpose through shared memory, one RED.ADD.F32x2 per (slice, k); the
// strays are worked off with global atomics, thread t taking moment t & 7 of stray t >> 3.  A pulse whose strays would
// not fit the list sorts the tile again (and is redone if they did not fit; after a sort at the pulse itself the
// overflow -- echoes outside the tile's slice window -- goes straight to global atomics, so the redo happens at most
// once).  Payload and stray list are double-buffered.
// Tried and measured in round 2 (profiles/r2_k2k_history.md): 512 threads x 2 facets with one CTA per SM, stage C by
// one thread per chunk of slots, producer / consumer warps behind named barriers, 2 and 4 facets per thread -- each
// cut the instruction count and none the time: with one CTA per SM the warps that sum the slices hold the others at
// the barrier, and at 4 facets per thread the state spills.
//
// Bound: issue slots (FP32 + integer mix); HBM/L2: four surface rows per facet and INTERVAL, the maps once.
#include <cstdio>

#include "kernels.cuh"
#include "geometry_common.cuh"

namespace heeps {

namespace {

constexpr int kKt = kMomentOrder;
static_assert(kKt == 8, "the sign pattern of the moment recurrence below is written for 8 moments");

constexpr int kRhoBias = 32768;           // slices added to rho so that it stays positive (unsigned 64-bit product)

struct __align__(16) KeyPulse {          // per pulse of the interval (shared memory)
    long long w;                         // (r0[p] - R_base) fs/c0 in 2^-48 slices
    uint32_t phi;                        // frac((r0[p] - R_base) / lambda) in 2^-32 turns
    float s;                             // (t - t0) / h
    int32_t base[kMaxKeyChannels];       // first slice of the tile's shared-memory window, per channel
};

// Exact state of one facet at one keyframe pulse.
struct KeyEval {
    double R, Rd;                        // path to the un-offset phase centre and its time derivative
    double la, lb;                       // r_r,c - r_r,ref = o_c la + o_c^2 lb  (series in o_c / r)
    double uat, uet, uar, uer, uao, ueo; // direction cosines: Tx azimuth / elevation, Rx (un-offset), Rx at the offset o_fd
};

__device__ __forceinline__ KeyEval key_eval(const PulseConst &pc, const double pos[3], const double vel[3], double o_fd)
{
    KeyEval o;
    const LegParts lt = leg_parts(pos, pc.tx_pos, pc.tx_a, pc.tx_e);
    const LegParts lr = leg_parts(pos, pc.rx_ref, pc.rx_a, pc.rx_e);
    o.R = lt.r + lr.r;
    const double at = fma(lt.dx, vel[0] - pc.tx_vel[0], fma(lt.dy, vel[1] - pc.tx_vel[1], lt.dz * (vel[2] - pc.tx_vel[2])));
    const double ar = fma(lr.dx, vel[0] - pc.rx_vel[0], fma(lr.dy, vel[1] - pc.rx_vel[1], lr.dz * (vel[2] - pc.rx_vel[2])));
    o.Rd = fma(at, lt.inv, ar * lr.inv);
    o.uat = lt.da * lt.inv; o.uet = lt.de * lt.inv; o.uar = lr.da * lr.inv; o.uer = lr.de * lr.inv;
    const double dv = fma(lr.dx, pc.rx_vhat[0], fma(lr.dy, pc.rx_vhat[1], lr.dz * pc.rx_vhat[2]));
    {
        double r_c, inv_c, da_c, de_c;
        channel_leg_series(lr, dv, o_fd, pc.rx_va, pc.rx_ve, r_c, inv_c, da_c, de_c);
        o.uao = da_c * inv_c; o.ueo = de_c * inv_c;
    }
    // r_c - r = r (dl/2 - dl^2/8 + ...), dl = (o^2 - 2 o d.v^)/r^2  (geometry_common.cuh)
    //         = -o (d.v^)/r + o^2 (1 - (d.v^/r)^2)/(2 r) + O(o^3/r^2)
    const double cv = dv * lr.inv;
    o.la = -cv;
    o.lb = 0.5 * lr.inv * fma(-cv, cv, 1.0);
    return o;
}

constexpr int kSplitMin = 48;             // stage C: an item with fewer echoes is not split between two teams
constexpr int kStrayCap = 96;             // stray echoes of one pulse held in shared memory (more: the tile is sorted again)
constexpr int kScrRow = 9;                // float2 per thread row of the transposition scratch (8 moments + 1 pad)
constexpr int kScrTeam = 8 * kScrRow;     // float2 per 8-thread team
__host__ __device__ constexpr int hist_words(int C, int span) { return (C * (span + 1) + 3) & ~3; }

// Packed f32x2 arithmetic on 64-bit registers (FFMA2 / FADD2): the operands stay register pairs from the
// shared-memory load to the transposition store, no pack / unpack moves in the moment loop.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float x, float y)
{
    f32x2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(x), "f"(y));
    return d;
}
__device__ __forceinline__ void unpk(f32x2 v, float &x, float &y)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(v));
}
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 fadd2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

__device__ __forceinline__ float pattern_x(float xa, float xe) { return sinc_pi_fast(xa) * sinc_pi_fast(xe); }

// Complex gain of antenna k at direction cosines (ua, ue): the table if there is one, else the analytic aperture.
template <bool kLut>
__device__ __forceinline__ float2 gain_at(const DevParams &prm, int k, double ua, double ue)
{
    if (kLut && prm.lut[k].tab) return lut_gain(prm.lut[k], ua, ue);
    const double apa = k ? prm.ap_rx_a : prm.ap_tx_a, ape = k ? prm.ap_rx_e : prm.ap_tx_e;
    return make_float2(pattern_x((float)(apa * ua), (float)(ape * ue)), 0.f);
}

// Coefficients (c1, c2, c3) of the cubic through (0, v0), (1/3, va), (2/3, vb), (1, v1); c0 = v0.
__device__ __forceinline__ void cubic_through(float v0, float va, float vb, float v1, float &c1, float &c2, float &c3)
{
    c1 = 0.5f * (-11.f * v0 + 18.f * va - 9.f * vb + 2.f * v1);
    c2 = 4.5f * (2.f * v0 - 5.f * va + 4.f * vb - v1);
    c3 = 4.5f * (-v0 + 3.f * va - 3.f * vb + v1);
}

// Slice word of a facet-echo: rho of the reference path at pulse index n ahead of the running state (Newton's forward
// formula; sort time only).
__device__ __forceinline__ unsigned long long rho_ahead(unsigned long long f, long long d1, long long d2, int d3, int n)
{
    const long long n1 = n, n2 = (long long)n * (n - 1) / 2, n3 = (long long)n * (n - 1) * (n - 2) / 6;
    return f + (unsigned long long)(n1 * d1 + n2 * d2 + n3 * (long long)d3);
}

constexpr int kThreads = 256;
// entries of stage C's work list: one per slice and channel, at least one per 8-thread team (split slices), even
__host__ __device__ constexpr int item_words(int C, int span)
{
    return ((C * (span + 1) > kThreads / 8 ? C * (span + 1) : kThreads / 8) + 1) & ~1;
}

// Checked build (python -m paper_2405_09938_b200.build --checked: -DHEEPS_CHECKED, libheeps_sim_checked.so): every
// computed shared-memory position and global moment-row index of this kernel is tested and a violation traps (the
// launch fails with a CUDA error).  compute-sanitizer is not available on the GPU pool this was developed on; the
// checked library runs tests/sanitizer_driver.py in its place.
#ifdef HEEPS_CHECKED
#define HEEPS_CHECK(cond) do { if (!(cond)) { printf("HEEPS_CHECK failed: %s (line %d, block %d, thread %d)\n", #cond, __LINE__, (int)blockIdx.x, (int)threadIdx.x); __trap(); } } while (0)
#else
#define HEEPS_CHECK(cond) do { } while (0)
#endif

// kDbg: the instantiation behind sim_debug_echoes, which also reports one pulse's facet-echoes.  A template flag and not
// a run-time test: the extra copy of the echo code inside the pulse loop cost the normal kernel 12 % (register
// allocation: 748 -> 854 ms on the Large configuration).
template <int FPT, int C, bool kTilt, bool kSpeckleT, bool kLut, bool kDbg>
__global__ void __launch_bounds__(kThreads, 2)
moments_keyframed_kernel(DevParams prm, MomentArgs a, int p0, int n_pl, int j_first)
{
    constexpr int NT = kThreads;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ PulseConst pc2[2];
    __shared__ KeyPulse s_kp[kMaxKeyPulses];
    __shared__ double s_rc[2][kMaxKeyChannels];          // path length of the tile centre at the two keyframes
    __shared__ double s_la_tile, s_lb_tile;              // a, b of the receive-channel series at the tile centre, first keyframe
    __shared__ int s_kept;
    __shared__ int s_rng[kMaxKeyChannels][2];
    __shared__ float4 s_stray[2][kStrayCap];                     // echoes that have left their sorted slice: (w, y, row index)
    __shared__ int s_nstray[3];
    __shared__ int s_blo[kMaxKeyChannels], s_bhi[kMaxKeyChannels];   // slices this tile touches during the interval
    __shared__ int s_dlamax;                                     // max |a - a_tile| + |a(t1) - a(t0)| over the tile, as float bits
    __shared__ int s_nitems;

    const int span = a.span_cap, hstride = span + 1;
    const int cap = prm.k2k_cap;
    const int capT = C * cap + 2;                        // slots of one payload buffer: C x cap, + the store target of echoes without a slot
    // [2][capT] float2 weight | [2][capT] float y | [C][cap] u32 slot of every facet-echo | [C][span + 1] int histogram |
    // [kThreads / 8][kScrTeam] float2 transposition scratch of stage C (+ the threads' stray stashes) | stage C work list |
    // [3][kThreads] float2 (am1, am2) | [3][kThreads] float2 (pq2, pq3): per-facet polynomial coefficients that are read
    // once per facet and pulse and would otherwise be spilled (128 registers at 2 CTAs per SM)
    float2 *payload = reinterpret_cast<float2 *>(smem_raw);
    float *payload_y = reinterpret_cast<float *>(smem_raw + (size_t)2 * capT * 8);
    uint32_t *slots = reinterpret_cast<uint32_t *>(smem_raw + (size_t)2 * capT * 12);
    int *hist = reinterpret_cast<int *>(smem_raw + (size_t)2 * capT * 12 + (size_t)C * cap * 4);
    float2 *scratch = reinterpret_cast<float2 *>(smem_raw + (size_t)2 * capT * 12 + (size_t)C * cap * 4 + (size_t)hist_words(C, span) * 4);
    // work list of stage C, written at every sort: one item per slice of [smin, smax) of every channel, channels end to end:
    // {first slot | echoes << 13 (0: empty, or outside the sampling window), channel | moment-row index << 2}
    uint2 *items = reinterpret_cast<uint2 *>(scratch + (kThreads / 8) * kScrTeam);
    float2 *amc = reinterpret_cast<float2 *>(items + item_words(C, span));   // [FPT][kThreads] tilt-modulation coefficients
    float2 *pqc = amc + 3 * kThreads;                                    // [FPT][kThreads] (pq2, pq3) of the gain cubic
    const uint32_t no_slot = (0x7ffffu << 13) | (uint32_t)(C * cap);      // slice 0x7ffff (never matches), store target = the spare slot

    const int tile = blockIdx.x, j = j_first + blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31;
    const int H = a.surf.H, P = a.surf.n_pulses_total;
    const int n_keys = (P - 1 + H - 1) / H + 1;
    const int k0 = min(j * H, P - 1), k1 = min((j + 1) * H, P - 1);
    // pulses of this interval inside the batch: [lo, hi)
    const int lo = max(j * H, p0), hi = min((j == n_keys - 2) ? P : (j + 1) * H, p0 + n_pl);
    if (lo >= hi) return;
    {
        const double *s0 = reinterpret_cast<const double *>(a.pulses + k0);
        const double *s1 = reinterpret_cast<const double *>(a.pulses + k1);
        double *d0 = reinterpret_cast<double *>(&pc2[0]), *d1 = reinterpret_cast<double *>(&pc2[1]);
        for (int k = tid; k < (int)(sizeof(PulseConst) / sizeof(double)); k += NT) { d0[k] = s0[k]; d1[k] = s1[k]; }
    }
    if (tid == 0) { s_kept = 0; s_nstray[0] = s_nstray[1] = s_nstray[2] = 0; s_dlamax = 0; s_nitems = 0; }
    if (tid < kMaxKeyChannels) { s_blo[tid] = 0x7fffffff; s_bhi[tid] = (int)0x80000000; }
    for (int k = tid; k < C * hstride; k += NT) hist[k] = 0;
    __syncthreads();

    // SHEARED TILES.  A tile is TH lines of TW facets; line b is displaced by rint(shear b) facets along the line
    // direction so that the lines' facets of equal index sit on one iso-range line (sim_create takes shear from the
    // path-length gradient at the scene centre): the tile spans TW |gradient along the line| range slices instead
    // of TW |g_a| + TH |g_b| -- three times fewer, fuller slices on the ATI geometry (8 instead of 27 per channel), so
    // three times less per-slice work in stage C and as many fewer RED.  axis 0: lines are grid rows (j), displaced in
    // i; axis 1: lines are grid columns (i), displaced in j.
    const int TW = prm.k2k_w, TH = prm.k2k_h, ltw = 31 - __clz(TW);
    const int ta0 = (tile % prm.k2k_tiles_a) * TW + prm.k2k_a0, tb0 = (tile / prm.k2k_tiles_a) * TH;
    auto facet_of = [&](int la, int lb, int &i, int &jj) {
        const int a_ = ta0 + la + __double2int_rn(prm.k2k_shear * (double)lb), b_ = tb0 + lb;
        i = prm.k2k_axis ? b_ : a_; jj = prm.k2k_axis ? a_ : b_;
    };
    if (tid < 2 * C) {
        // tile centre (rest height, advected by the current at the centre facet) at the two keyframes: positions the
        // slice window of every pulse between; and the receive-channel series there (a, b at the first keyframe)
        const int e = tid / C, c = tid - e * C;
        const PulseConst &pc = pc2[e];
        int ici, jci;
        facet_of(TW / 2, TH / 2, ici, jci);
        ici = min(max(ici, 0), prm.nx - 1); jci = min(max(jci, 0), prm.ny - 1);      // (a tile at the grid's edge: nearest facet)
        double cux = prm.cur_ux, cuy = prm.cur_uy;
        if (a.current) {
            const float2 cv = __ldg(a.current + (size_t)jci * prm.nx + ici);
            cux = cv.x; cuy = cv.y;
        }
        const double x = prm.cx + ((double)ici - 0.5 * (prm.nx - 1)) * prm.spacing + cux * pc.t;
        const double y = prm.cy + ((double)jci - 0.5 * (prm.ny - 1)) * prm.spacing + cuy * pc.t;
        const double ax = x - pc.tx_pos[0], ay = y - pc.tx_pos[1], az = prm.cz - pc.tx_pos[2];
        const double bx = x - pc.rx_pos[c][0], by = y - pc.rx_pos[c][1], bz = prm.cz - pc.rx_pos[c][2];
        s_rc[e][c] = sqrt(ax * ax + ay * ay + az * az) + sqrt(bx * bx + by * by + bz * bz);
        if (tid == 0) {
            const double dx = x - pc.rx_ref[0], dy = y - pc.rx_ref[1], dz = prm.cz - pc.rx_ref[2];
            const double inv = rsqrt(dx * dx + dy * dy + dz * dz);
            const double cv = (dx * pc.rx_vhat[0] + dy * pc.rx_vhat[1] + dz * pc.rx_vhat[2]) * inv;
            s_la_tile = -cv; s_lb_tile = 0.5 * inv * (1.0 - cv * cv);
        }
    }
    __syncthreads();
    const double Rbase = pc2[0].r0;                              // c0 t0 of the first keyframe
    const double two48 = 281474976710656.0;
    for (int ip = tid; ip < hi - lo; ip += NT) {
        const int p = lo + ip;
        const double t0 = pc2[0].t, t1 = pc2[1].t, t = a.pulses[p].t;
        const double h = t1 - t0;
        const double s = (h != 0.0) ? (t - t0) / h : 0.0;
        const double r0 = a.pulses[p].r0;
        KeyPulse kp;
        kp.w = __double2ll_rn((r0 - Rbase) * prm.fs_over_c0 * two48);
        kp.phi = turns_to_u32_fast((r0 - Rbase) * prm.inv_lambda);
        kp.s = (float)s;
#pragma unroll
        for (int c = 0; c < kMaxKeyChannels; ++c) {
            int base = 0;
            if (c < C) {
                const double rc = fma(s, s_rc[1][c] - s_rc[0][c], s_rc[0][c]);
                double bc = ceil((rc - r0) * prm.fs_over_c0 - prm.half_len) - 0.5 * span;
                bc = fmin(fmax(bc, -1.0e9), 1.0e9);
                base = (int)bc;
            }
            kp.base[c] = base;
        }
        s_kp[ip] = kp;
    }

    // ---- interpolants of this thread's facets over the interval ----
    const size_t F = (size_t)prm.nx * prm.ny;
    const size_t row0 = (size_t)(j - a.surf.key0) * F, row1 = row0 + F;
    const float area = (float)(prm.spacing * prm.spacing);
    double o_fd = 0.0;
#pragma unroll
    for (int c = 0; c < C; ++c) o_fd = fmax(o_fd, fabs(pc2[0].ch_off[c]));
    const float inv_ofd = (o_fd > 0.0) ? (float)(1.0 / o_fd) : 0.f;
    const int n_int = max(k1 - k0, 1), i0 = lo - k0;                // pulses of the interval; index of this CTA's first pulse
    const double la_tile = s_la_tile;

    unsigned long long rho[FPT];                                     // path of the facet at the current pulse (2^-48 slices, < 2^16 slices)
    long long rd1[FPT], rd2[FPT];                                    // its running forward differences
    int rd3[FPT];
    float dla0[FPT], dla[FPT];                                       // a(t0) - a_tile, a(t1) - a(t0)  (set-up: as computed; then scaled, see dG below)
    float pq0[FPT], pq1[FPT], pq2[FPT], pq3[FPT], bq[FPT];           // P(s) = pq0 + s (pq1 + s (pq2 + s pq3)); bq = G_t dG_r/do
    constexpr int FL = kLut ? FPT : 1;                               // tabulated patterns: P and bq are complex, the imaginary parts
    float qi0[FL], qi1[FL], qi2[FL], qi3[FL], bqi[FL];
    float am0[FPT];
    // |a_f|(s) = am0 + s (am1 + s am2) when tilt-modulated: (am1, am2) of the thread's facets live in shared memory
    // (amc[q][tid], one LDS.64 per facet and pulse; six registers less in the pulse loop)
    uint32_t xarg[FPT];
    int fidx[kSpeckleT ? FPT : 1];                                   // facet index (time-dependent speckle: one load per pulse)
    unsigned validmask = 0;
    float my_dla = 0.f;
#pragma unroll
    for (int q = 0; q < FPT; ++q) {
        const int k = q * NT + tid;
        int i, jj;
        facet_of(k & (TW - 1), k >> ltw, i, jj);
        const bool valid = (k < TW * TH && i >= 0 && i < prm.nx && jj >= 0 && jj < prm.ny);
        if (kSpeckleT) fidx[kSpeckleT ? q : 0] = valid ? jj * prm.nx + i : 0;
        rho[q] = (unsigned long long)kRhoBias << 48; rd1[q] = rd2[q] = 0; rd3[q] = 0;
        dla0[q] = dla[q] = 0.f;
        pq0[q] = pq1[q] = pq2[q] = pq3[q] = bq[q] = 0.f; am0[q] = 0.f; xarg[q] = 0u;
        if (kLut) qi0[q] = qi1[q] = qi2[q] = qi3[q] = bqi[q] = 0.f;
        if (kTilt) amc[q * NT + tid] = make_float2(0.f, 0.f);
        if (!valid) continue;
        const size_t f = (size_t)jj * prm.nx + i;
        const double xb = prm.cx + ((double)i - 0.5 * (prm.nx - 1)) * prm.spacing;
        const double yb = prm.cy + ((double)jj - 0.5 * (prm.ny - 1)) * prm.spacing;
        double cux = prm.cur_ux, cuy = prm.cur_uy;
        if (a.current) { const float2 cv = __ldg(a.current + f); cux = cv.x; cuy = cv.y; }
        KeyEval ev[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const PulseConst &pc = pc2[e];
            const size_t r = (e ? row1 : row0) + f;
            double pos[3] = {fma(cux, pc.t, xb), fma(cuy, pc.t, yb), prm.cz + a.surf.z[r]};
            double vel[3] = {cux, cuy, a.surf.zt[r]};
            if (a.surf.dxy) {
                const double2 dd = a.surf.dxy[r], dt = a.surf.dxy_t[r];
                pos[0] += dd.x; pos[1] += dd.y; vel[0] += dt.x; vel[1] += dt.y;
            }
            ev[e] = key_eval(pc, pos, vel, o_fd);
        }
        {
            // Hermite cubic of the path in the pulse index i (uniform pulse times):  R(i) = R0 + a1 i + a2 i^2 + a3 i^3,
            // ra = h R0' - D, rb = h R1' - D, D = R1 - R0;  in range slices, and its forward differences at i0
            const double hh = pc2[1].t - pc2[0].t, D = ev[1].R - ev[0].R;
            const double ra = fma(hh, ev[0].Rd, -D), rb = fma(hh, ev[1].Rd, -D);
            const double inv_n = 1.0 / (double)n_int, fsc = prm.fs_over_c0;
            const double c0q = fma(ev[0].R - Rbase, fsc, (double)kRhoBias - prm.half_len);
            const double c1 = (D + ra) * fsc * inv_n, c2 = (-2.0 * ra - rb) * fsc * inv_n * inv_n;
            const double c3 = (ra + rb) * fsc * inv_n * inv_n * inv_n;
            const double x0 = (double)i0;
            const double f0 = fma(x0, fma(x0, fma(x0, c3, c2), c1), c0q);
            const double g1 = c1 + c2 * (2.0 * x0 + 1.0) + c3 * (3.0 * x0 * x0 + 3.0 * x0 + 1.0);
            const double g2 = 2.0 * c2 + c3 * (6.0 * x0 + 6.0), g3 = 6.0 * c3;
            if (f0 > 64.0 && f0 < 65536.0 - 64.0 && fabs(g1) < 0.5) {   // inside the fixed-point range (else: no echo; the host guard keeps scenes inside)
                rho[q] = __double2ull_rn(f0 * two48); rd1[q] = __double2ll_rn(g1 * two48);
                rd2[q] = __double2ll_rn(g2 * two48); rd3[q] = (int)__double2ll_rn(g3 * two48);
                validmask |= 1u << q;
            }
        }
        dla0[q] = (float)(ev[0].la - la_tile);
        dla[q] = (float)(ev[1].la - ev[0].la);
        my_dla = fmaxf(my_dla, fabsf(dla0[q]) + fabsf(dla[q]));
        // gains at s = 0, 1/3, 2/3, 1 (direction cosines between the keyframes interpolated linearly)
        {
            float2 Pn[4];
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                const double sn = n * (1.0 / 3.0);
                const float2 gt = gain_at<kLut>(prm, 0, fma(sn, ev[1].uat - ev[0].uat, ev[0].uat), fma(sn, ev[1].uet - ev[0].uet, ev[0].uet));
                const float2 gr = gain_at<kLut>(prm, 1, fma(sn, ev[1].uar - ev[0].uar, ev[0].uar), fma(sn, ev[1].uer - ev[0].uer, ev[0].uer));
                Pn[n] = kLut ? cmulf(gt, gr) : make_float2(gt.x * gr.x, 0.f);
            }
            const float2 gtm = gain_at<kLut>(prm, 0, 0.5 * (ev[0].uat + ev[1].uat), 0.5 * (ev[0].uet + ev[1].uet));
            const float2 grm = gain_at<kLut>(prm, 1, 0.5 * (ev[0].uar + ev[1].uar), 0.5 * (ev[0].uer + ev[1].uer));
            const float2 gom = gain_at<kLut>(prm, 1, 0.5 * (ev[0].uao + ev[1].uao), 0.5 * (ev[0].ueo + ev[1].ueo));
            pq0[q] = Pn[0].x;
            cubic_through(Pn[0].x, Pn[1].x, Pn[2].x, Pn[3].x, pq1[q], pq2[q], pq3[q]);
            if (kLut) {
                qi0[q] = Pn[0].y;
                cubic_through(Pn[0].y, Pn[1].y, Pn[2].y, Pn[3].y, qi1[q], qi2[q], qi3[q]);
                const float2 dq = cmulf(gtm, make_float2((gom.x - grm.x) * inv_ofd, (gom.y - grm.y) * inv_ofd));
                bq[q] = dq.x; bqi[q] = dq.y;
            } else {
                bq[q] = gtm.x * (gom.x - grm.x) * inv_ofd;
            }
        }
        // amplitude (O8): sqrt(sigma0 tilt d^2) |xi|
        const float sig = a.sigma0 ? __ldg(a.sigma0 + f) : (float)prm.sigma0_uniform;
        // static speckle: |xi| and arg xi are constants of the facet; time-dependent speckle (speckle.cu): per pulse
        float xmag = 1.f;
        if (!kSpeckleT) { const uint2 xp = __ldg(a.xi_polar + f); xmag = __uint_as_float(xp.x); xarg[q] = xp.y; }
        if (kTilt) {
            const float2 sl0 = a.surf.slope[row0 + f], sl1 = a.surf.slope[row1 + f];
            float2 slm = make_float2(0.5f * (sl0.x + sl1.x), 0.5f * (sl0.y + sl1.y));   // slopes are linear between keyframes ...
            if (a.surf.slope_t) {                                // ... or cubic Hermite: value at mid-interval = mean + h (s0' - s1') / 8
                const float2 r0 = a.surf.slope_t[row0 + f], r1 = a.surf.slope_t[row1 + f];
                const float h8 = 0.125f * (float)(pc2[1].t - pc2[0].t);
                slm.x = fmaf(h8, r0.x - r1.x, slm.x); slm.y = fmaf(h8, r0.y - r1.y, slm.y);
            }
            const float lx = (float)prm.look_x, ly = (float)prm.look_y;
            const float A0 = sqrtf(sig * fmaxf(1.f + 2.f * (sl0.x * lx + sl0.y * ly), 0.f) * area) * xmag;
            const float Am = sqrtf(sig * fmaxf(1.f + 2.f * (slm.x * lx + slm.y * ly), 0.f) * area) * xmag;
            const float A1 = sqrtf(sig * fmaxf(1.f + 2.f * (sl1.x * lx + sl1.y * ly), 0.f) * area) * xmag;
            am0[q] = A0; amc[q * NT + tid] = make_float2(-3.f * A0 + 4.f * Am - A1, 2.f * A0 - 4.f * Am + 2.f * A1);
        } else {
            am0[q] = sqrtf(sig * area) * xmag;
        }
    }
    if (my_dla > 0.f) atomicMax(&s_dlamax, __float_as_int(my_dla));
    __syncthreads();                                     // s_kp, s_dlamax complete

    // ---- per-channel constants ----
    const int L = a.replica;
    const unsigned win_hi = (unsigned)(prm.n_samples + L - 1);
    float och[C];
    float och_max = 0.f;
#pragma unroll
    for (int c = 0; c < C; ++c) {
        och[c] = (float)pc2[0].ch_off[c];
        och_max = fmaxf(och_max, fabsf(och[c]));
    }
    // The receive-channel path difference o_c a + o_c^2 b with a = a_tile + (a_f(t0) - a_tile) + s (a_f(t1) - a_f(t0)):
    // the tile-centre part is one exact word per channel for the phase (2^-32 turns) and one for the slice (2^-32
    // slices); the facet's part, -o_c (...) / lambda in units of `mult` 2^-32 turns, is kept under 2^21 so that one FFMA
    // against 1.5 x 2^23 rounds it to an integer in the mantissa (likewise o_c (...) fs/c0 in 2^-32 slices: smaller).
    const double il32 = prm.inv_lambda * 4294967296.0;
    uint32_t mult = 1;
    {
        const float lin_max = och_max * __int_as_float(s_dlamax) * (float)il32;
        while ((float)mult * 2097152.f < lin_max && mult < (1u << 20)) mult <<= 1;
    }
    uint32_t PSI[C], DNU[C];
#pragma unroll
    for (int c = 0; c < C; ++c) {
        const double o = pc2[0].ch_off[c];
        const double dl_tile = o * fma(o, s_lb_tile, la_tile);           // r_r,c - r_r,ref at the tile centre, first keyframe [m]
        PSI[c] = turns_to_u32_fast(-dl_tile * prm.inv_lambda) + prm.phase_bias32 - 0x4B400000u * mult;
        DNU[c] = (uint32_t)__double2int_rn(dl_tile * prm.fs_over_c0 * 4294967296.0) - 0x4B400000u;
    }
    // facet part: g(s) = dG0 + s dGs in units of mult 2^-32 turns per metre of offset; in 2^-32 slices: g(s) x slice_per_g
    const float to_g = -(float)il32 / (float)mult;
    const float slice_per_g = -(float)mult * (float)(prm.fs_over_c0 / prm.inv_lambda);
#pragma unroll
    for (int q = 0; q < FPT; ++q) { dla0[q] *= to_g; dla[q] *= to_g; }    // now dG0, dGs

#pragma unroll
    for (int q = 0; q < FPT; ++q) pqc[q * NT + tid] = make_float2(pq2[q], pq3[q]);
    int my_kept = 0;
    const int sub = tid & 7, team = tid >> 3, warp = tid >> 5;
    float2 *scr = scratch + team * kScrTeam;
    // the thread's stray stash: C float4 inside its team's transposition scratch (stage C of the same warp uses the
    // scratch only after this pulse's barrier, the stash is written and read before it); quarter-warp conflict-free
    static_assert((size_t)kScrTeam * sizeof(float2) >= 8 * (size_t)C * sizeof(float4) + 16, "stash does not fit the team scratch");
    float4 *stash = reinterpret_cast<float4 *>((reinterpret_cast<uintptr_t>(scr) + 15) & ~(uintptr_t)15) + sub * C;
    const int capS = C * cap;                                            // slots of all channels (the spare one follows)

    // ---- The facet-echoes of the tile are ordered by range slice ONCE (counting sort at the interval's middle pulse:
    //      histogram by integer ATOMS, scan, slot = first position of the slice + rank), not at every pulse: over the
    //      few milliseconds of an interval a facet's slice changes only when its sub-slice position crosses 0 or 1
    //      (the window follows the scene: a percent or two of the echoes per pulse).  At every pulse an echo found in
    //      its sorted slice writes its weight into its slot; one found elsewhere ("stray") leaves a zero there and goes
    //      to a short shared-memory list that the CTA works off with global atomics.  A pulse with more strays than the
    //      list holds sorts the tile again at that pulse and is redone.  Stage C reads each slice's slots
    //      contiguously: no per-pulse histogram, scan or index list; one barrier per pulse. ----
    int *hs = hist;                                                  // [C][span + 1] first slot of each slice
    int K2[C];                                                       // slice index relative to the tile window = (word >> 32) - K2[c]
#pragma unroll
    for (int c = 0; c < C; ++c) K2[c] = 0;
    int ip_sort = (hi - lo) / 2;
    {
        const double drift = fabs((s_rc[1][0] - s_rc[0][0]) - (a.pulses[k1].r0 - a.pulses[k0].r0)) * prm.fs_over_c0 /
                             (double)max(k1 - k0, 1);
        if (drift * (double)(TW * TH * C) * 0.5 * (double)(hi - lo) > 0.9 * kStrayCap) ip_sort = 0;
    }
    bool need_sort = true;
    int ns_prev = 0;                                                 // strays of the previous pulse (0 after a sort)
    int sorted_at = -1;
    int ns_cur = 0;                                                  // which of the three stray counters this pulse uses

    // slice word of facet q, channel c at pulse state (X = reference path, s): [slice + kRhoBias . fraction]
    auto slice_word = [&](int q, int c, long long X, float nq) -> long long {
        const float t3 = fmaf(och[c], nq, 12582912.f);
        return X + (long long)(int32_t)(DNU[c] + __float_as_uint(t3));
    };

    for (int ip = 0; ip < hi - lo;) {
        if (need_sort) {
            need_sort = false;
            sorted_at = ip_sort;
            const KeyPulse &kps = s_kp[ip_sort];
            __syncthreads();                                         // nobody reads the old histogram / slots any more
            for (int k = tid; k < C * hstride; k += NT) hs[k] = 0;
            if (tid == 0) s_nstray[ns_cur] = 0;
            __syncthreads();
            int bref[C];
#pragma unroll
            for (int c = 0; c < C; ++c) { bref[c] = kps.base[c]; K2[c] = bref[c] + kRhoBias - 1; }
            int pr[FPT][C];
#pragma unroll
            for (int q = 0; q < FPT; ++q) {
                const long long X = (long long)((rho_ahead(rho[q], rd1[q], rd2[q], rd3[q], ip_sort - ip) - (unsigned long long)kps.w) >> 16);
                const float nq = fmaf(kps.s, dla[q], dla0[q]) * slice_per_g;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    const int rel = (int)(slice_word(q, c, X, nq) >> 32) - K2[c];
                    pr[q][c] = -1;
                    if (((validmask >> q) & 1u) && (unsigned)rel < (unsigned)span)
                    {
                        HEEPS_CHECK(rel + 1 <= span);
                        pr[q][c] = (rel << 12) | atomicAdd(&hs[c * hstride + rel + 1], 1);
                    }
                }
            }
            __syncthreads();
            if (warp < C) {                                          // inclusive scan: hs[c][s] = first slot of slice s
                int *hc = hs + warp * hstride;
                int carry = 0, smin = span, smax = 0;
                for (int k0s = 1; k0s <= span; k0s += 32) {
                    const int k = k0s + lane;
                    int v = (k <= span) ? hc[k] : 0;
                    if (v > 0) { smin = min(smin, k - 1); smax = max(smax, k); }
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int t = __shfl_up_sync(0xffffffffu, v, o);
                        if (lane >= o) v += t;
                    }
                    if (k <= span) hc[k] = v + carry;
                    carry += __shfl_sync(0xffffffffu, v, 31);
                }
                smin = __reduce_min_sync(0xffffffffu, smin);
                smax = __reduce_max_sync(0xffffffffu, smax);
                if (lane == 0) {
                    s_rng[warp][0] = smin; s_rng[warp][1] = smax;                      // occupied slices [smin, smax)
                    if (smax > smin) {                                                 // the band this tile reports to K3s
                        atomicMin(&s_blo[warp], bref[warp] + smin - 1); atomicMax(&s_bhi[warp], bref[warp] + smax + 1);
                    }
                }
            }
            __syncthreads();
            {
                int pre[C + 1];                                            // first item of channel c
                pre[0] = 0;
#pragma unroll
                for (int c = 0; c < C; ++c) pre[c + 1] = pre[c] + max(s_rng[c][1] - s_rng[c][0], 0);
                const int total = pre[C];
                if (tid == 0) s_nitems = total;
                for (int it = tid; it < total; it += NT) {
                    int c = 0;
#pragma unroll
                    for (int cc = 1; cc < C; ++cc) c = (it >= pre[cc]) ? cc : c;
                    int pc0 = 0, bc = bref[0];
#pragma unroll
                    for (int cc = 1; cc < C; ++cc) { pc0 = (c == cc) ? pre[cc] : pc0; bc = (c == cc) ? bref[cc] : bc; }
                    const int sidx = s_rng[c][0] + (it - pc0);
                    const int first = hs[c * hstride + sidx];
                    int cnt = hs[c * hstride + sidx + 1] - first;
                    const int jb = bc + sidx + L - 1;                      // slice b = bref + sidx sits at row index b + L - 1
                    if ((unsigned)jb >= win_hi) cnt = 0;                   // a slice outside the sampling window holds zeros only
                    HEEPS_CHECK(cnt == 0 || (first >= 0 && first + cnt <= cap && jb < a.nb_pad));
                    items[it] = make_uint2((uint32_t)(c * cap + first) | ((uint32_t)cnt << 13), (uint32_t)c | ((uint32_t)max(jb, 0) << 2));
                }
                // Fewer slices than 8-thread teams (a tile of the Large configuration: 18 slices of up to 220 echoes for 32
                // teams): the fullest item is halved until every team has one (the halves add into the same moment row; the
                // second half goes to the end of the list, i.e. to another warp).  The barrier of a pulse waits for the team
                // with the longest item: 2.0 barrier-stall cycles per issue on Large before this (round 2).  All items were
                // written by warp 0 when there are at most 32.
                if (warp == 0 && total < kThreads / 8) {
                    __syncwarp();
                    uint2 my = (lane < total) ? items[lane] : make_uint2(0u, 0u);
                    int n = total;
                    while (n < kThreads / 8) {
                        const unsigned best = __reduce_max_sync(0xffffffffu, ((my.x >> 13) << 5) | (unsigned)lane);
                        const int bc = (int)(best >> 5), bl = (int)(best & 31u);
                        if (bc < kSplitMin) break;
                        const int h = ((bc >> 1) + 7) & ~7;                // the first half keeps whole octets
                        const uint32_t sx = __shfl_sync(0xffffffffu, my.x, bl), sy = __shfl_sync(0xffffffffu, my.y, bl);
                        if (lane == bl) my.x = (sx & 8191u) | ((uint32_t)h << 13);
                        if (lane == n) { my.x = ((sx & 8191u) + (uint32_t)h) | ((uint32_t)(bc - h) << 13); my.y = sy; }
                        ++n;
                    }
                    // longest first: the four teams of a warp run their items in step, so a warp should hold items of like length
                    const unsigned mykey = ((my.x >> 13) << 5) | (unsigned)(31 - lane);
                    int rank = 0;
                    for (int o = 0; o < kThreads / 8; ++o) rank += (__shfl_sync(0xffffffffu, mykey, o) > mykey) ? 1 : 0;
                    if (lane < n) items[rank] = my;
                    if (lane == 0) s_nitems = n;
                }
            }
#pragma unroll
            for (int q = 0; q < FPT; ++q)
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    const int v = pr[q][c];
                    HEEPS_CHECK(v < 0 || ((v & 4095) < cap && hs[c * hstride + (v >> 12)] + (v & 4095) < cap));
                    if (FPT > 1 || q * NT + tid < cap)               // (FPT = 1: the tile may be smaller than the CTA)
                        slots[c * cap + q * NT + tid] =
                            (v >= 0) ? (uint32_t)(((v >> 12) << 13) | (c * cap + hs[c * hstride + (v >> 12)] + (v & 4095))) : no_slot;
                }
            // a thread reads only its own slots; the scan results are read after the barrier of stage A
        }
        const int buf = ip & 1;
        const int pl = lo + ip - p0;
        const KeyPulse kp = s_kp[ip];
        float2 *pay = payload + (size_t)buf * capT;
        float *pay_y = payload_y + (size_t)buf * capT;
        const float s = kp.s;
        int *n_stray = &s_nstray[ns_cur];
        const int ns_next = (ns_cur == 2) ? 0 : ns_cur + 1;
        if (tid == 0) s_nstray[ns_next] = 0;                 // last read two pulses ago, next written after this pulse's barrier
        int kept_p = 0;

        // ---- A: slice, sub-slice position, complex weight of every facet-echo, written to the echo's slot.
        //      Branch-free straight-line code for all FPT x C echoes of the thread, so that the independent chains
        //      (integer slice word -> MUFU -> stores) interleave.  A stray is written (one predicated STS.128) to the
        //      thread's stash and appended to the pulse's list after the loop; a thread's second stray of one channel
        //      in one pulse only sets a bit and is worked off after the loop by evaluating that echo again.  (Round 2:
        //      re-evaluating every stray was 11 % of the kernel's instructions on the Large configuration.)
        unsigned stray_mask = 0, stashed = 0;
        // sorted at this very pulse and still no room in the list: the stray's eight moments straight to the rows
        auto straight_to_the_rows = [&](const float4 e) {
            const int code = __float_as_int(e.w), c = code >> 28, jb = code & 0x0fffffff;
            float2 *row = a.mom + ((size_t)(c * n_pl + pl) * kKt) * a.nb_pad + jb;
            float t0 = 1.f, t1 = e.z;
            atomicAdd(row, make_float2(e.x, e.y));
            atomicAdd(row + a.nb_pad, make_float2(e.x * t1, e.y * t1));
            for (int k2 = 2; k2 < kKt; ++k2) {
                const float t2k = 2.f * e.z * t1 - t0;
                atomicAdd(row + (size_t)k2 * a.nb_pad, make_float2(e.x * t2k, e.y * t2k));
                t0 = t1; t1 = t2k;
            }
            const int b = jb - (L - 1);
            atomicMin(&s_blo[c], b); atomicMax(&s_bhi[c], b + 1);
        };
        auto facet = [&](const int q, float &Pv, float &Pi, float &am, uint32_t &ph_ref, long long &X, float &gq, bool &keep) {
            const float2 p23 = pqc[q * NT + tid];
            Pv = fmaf(s, fmaf(s, fmaf(s, p23.y, p23.x), pq1[q]), pq0[q]);
            Pi = kLut ? fmaf(s, fmaf(s, fmaf(s, qi3[kLut ? q : 0], qi2[kLut ? q : 0]), qi1[kLut ? q : 0]), qi0[kLut ? q : 0]) : 0.f;
            keep = ((validmask >> q) & 1u) && !(kLut ? (fmaf(Pv, Pv, Pi * Pi) < prm.cull_thr * prm.cull_thr)
                                                     : (fabsf(Pv) < prm.cull_thr));     // O7 (G6)
            am = am0[q];
            if (kTilt) { const float2 c12 = amc[q * NT + tid]; am = fmaf(s, fmaf(s, c12.y, c12.x), am); }
            uint32_t xa = xarg[q];
            if (kSpeckleT && ((validmask >> q) & 1u)) {   // time-dependent speckle: s_f(t_p) of this pulse (eq. (7), (10))
                const uint2 xp = __ldg(a.xi_polar + (size_t)pl * a.xi_pulse_stride + (size_t)fidx[kSpeckleT ? q : 0]);
                am *= __uint_as_float(xp.x); xa = xp.y;
            }
            am = keep ? am : 0.f;
            // carrier phase of the reference path: the 32 fraction bits of rho x (f0 / fs)
            const uint32_t r_lo = (uint32_t)rho[q], r_hi = (uint32_t)(rho[q] >> 32);
            const uint32_t T = __umulhi(r_lo, prm.ratio_hi) + __umulhi(r_hi, prm.ratio_lo) + r_hi * prm.ratio_hi;
            ph_ref = kp.phi - T + xa;
            X = (long long)((rho[q] - (unsigned long long)kp.w) >> 16);   // [slice + kRhoBias . 32-bit fraction], positive
            gq = fmaf(s, dla[q], dla0[q]);                                 // channel series of this facet at this pulse
        };
        auto echo = [&](const int q, const int c, const float Pv, const float Pi, const float am, const uint32_t ph_ref,
                        const long long X, const float gq, const float nq, float &wr, float &wi, float &yv, int &xh) {
            const long long Xc = slice_word(q, c, X, nq);
            xh = (int)(Xc >> 32);
            const uint32_t fr = (uint32_t)(unsigned long long)Xc;
            // b = ceil(nu) = xh + 1 - kRhoBias; eps = b - nu = 1 - fr 2^-32; y = 2 eps - 1 = 3 - 2 (1 + fr 2^-32)
            yv = fmaf(__uint_as_float(0x3F800000u | (fr >> 9)), -2.f, 3.f);
            const float t2 = fmaf(och[c], gq, 12582912.f);
            const uint32_t ph = PSI[c] + ph_ref + __float_as_uint(t2) * mult;
            float sn, cs;
            __sincosf((float)(int32_t)ph * 1.4629180792671596e-9f, &sn, &cs);   // 2 pi / 2^32
            const float g = fmaf(och[c], bq[q], Pv);
            if (kLut) {                                                    // complex gain times the phasor
                const float gi = fmaf(och[c], bqi[kLut ? q : 0], Pi);
                wr = am * fmaf(g, cs, -gi * sn); wi = am * fmaf(g, sn, gi * cs);
            } else {
                const float mag = g * am;
                wr = mag * cs; wi = mag * sn;
            }
        };
#pragma unroll
        for (int q = 0; q < FPT; ++q) {
            float Pv, Pi, am, gq; uint32_t ph_ref; long long X; bool keep;
            facet(q, Pv, Pi, am, ph_ref, X, gq, keep);
            const float nq = gq * slice_per_g;
            kept_p += keep ? 1 : 0;
            const int k = q * NT + tid;
#pragma unroll
            for (int c = 0; c < C; ++c) {
                float wr, wi, yv; int xh;
                echo(q, c, Pv, Pi, am, ph_ref, X, gq, nq, wr, wi, yv, xh);
                const uint32_t slot = (FPT > 1 || k < cap) ? slots[c * cap + k] : no_slot;
                const bool here = (uint32_t)(xh - K2[c]) == (slot >> 13);   // in its sorted slice
                const uint32_t pos = slot & 8191u;
                HEEPS_CHECK(pos <= (uint32_t)capS && (!here || pos < (uint32_t)capS));
                pay[pos] = here ? make_float2(wr, wi) : make_float2(0.f, 0.f);
                pay_y[pos] = yv;
                // stray: left its sorted slice, or never had one; its window meets [0, Ns).  The thread's first stray of a
                // channel goes to its stash (a facet that crosses a slice edge does so in every channel); any other sets a bit
                const int jb = xh + 1 - kRhoBias + (L - 1);
                const bool stray = !here && keep && ((unsigned)jb < win_hi);
                const bool first = stray && !((stashed >> c) & 1u);
                if (first) stash[c] = make_float4(wr, wi, yv, __int_as_float((c << 28) | jb));
                stray_mask |= (stray && !first) ? (1u << (q * C + c)) : 0u;
                stashed |= stray ? (1u << c) : 0u;
            }
        }
        if (stashed) {
#pragma unroll
            for (int c = 0; c < C; ++c) {
                if (!((stashed >> c) & 1u)) continue;
                const int t = atomicAdd(n_stray, 1);
                if (t < kStrayCap) s_stray[buf][t] = stash[c];
                else if (sorted_at == ip) straight_to_the_rows(stash[c]);
            }
        }
        if (stray_mask) {
#pragma unroll
            for (int q = 0; q < FPT; ++q) {
                if (((stray_mask >> (q * C)) & ((1u << C) - 1u)) == 0u) continue;
                float Pv, Pi, am, gq; uint32_t ph_ref; long long X; bool keep;
                facet(q, Pv, Pi, am, ph_ref, X, gq, keep);
                const float nq = gq * slice_per_g;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    if (!((stray_mask >> (q * C + c)) & 1u)) continue;
                    float wr, wi, yv; int xh;
                    echo(q, c, Pv, Pi, am, ph_ref, X, gq, nq, wr, wi, yv, xh);
                    const int b = xh + 1 - kRhoBias;
                    const int t = atomicAdd(n_stray, 1);
                    HEEPS_CHECK(b + L - 1 >= 0 && b + L - 1 < a.nb_pad);
                    const float4 e = make_float4(wr, wi, yv, __int_as_float((c << 28) | (b + L - 1)));
                    if (t < kStrayCap) s_stray[buf][t] = e;
                    else if (sorted_at == ip) straight_to_the_rows(e);
                }
            }
        }
        if (kDbg && a.dbg_slice && lo + ip == a.dbg_pulse) {  // sim_debug_echoes: this pulse's facet-echoes as the kernel sees them
#pragma unroll
            for (int q = 0; q < FPT; ++q) {
                const int k = q * NT + tid;
                int i, jj;
                facet_of(k & (TW - 1), k >> ltw, i, jj);
                if (!(k < TW * TH && i >= 0 && i < prm.nx && jj >= 0 && jj < prm.ny)) continue;
                const size_t f = (size_t)jj * prm.nx + i;
                float Pv, Pi, am, gq; uint32_t ph_ref; long long X; bool keep;
                facet(q, Pv, Pi, am, ph_ref, X, gq, keep);
                const float nq = gq * slice_per_g;
                a.dbg_keep[f] = keep ? 1 : 0;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    float wr, wi, yv; int xh;
                    echo(q, c, Pv, Pi, am, ph_ref, X, gq, nq, wr, wi, yv, xh);
                    a.dbg_slice[(size_t)c * F + f] = xh + 1 - kRhoBias;
                    a.dbg_eps[(size_t)c * F + f] = 0.5f * (yv + 1.f);
                    a.dbg_w[(size_t)c * F + f] = make_float2(wr, wi);
                }
            }
        }
        __syncthreads();
        const int ns_all = *n_stray;
        if (ns_all > kStrayCap && sorted_at != ip) {         // too many have moved on: sort the tile at this pulse, redo it
            need_sort = true; ip_sort = ip;
            continue;
        }
        const int ns = min(ns_all, kStrayCap);
        my_kept += kept_p;

        // ---- C: 8 threads per slice: Chebyshev moments over the slice's slots, transpose through shared memory, one
        //      RED per (slice, k).  The recurrence runs on a_k = sigma_k T_k, sigma = + + - - + + - -, which needs no
        //      negation: a_{k+1} = -+ 2y a_k + a_{k-1} (minus for odd k); sigma_k is applied to the slice sum.
        //      Work items = the occupied slices of all C channels laid end to end.
        {
            const int total = s_nitems;
            // moment row `sub` of this pulse, channel 0 (the channel adds c n_pl Kt rows)
            float2 *const row0 = a.mom + ((size_t)pl * kKt + sub) * a.nb_pad;
            const size_t cstride = (size_t)n_pl * kKt * a.nb_pad;
            for (int it0 = 0; it0 < total; it0 += kThreads / 8) {
                if (it0 + warp * 4 >= total) break;                        // warp-uniform
                const int it = it0 + team;
                const uint2 item = (it < total) ? items[it] : make_uint2(0u, 0u);
                const int cnt = (int)(item.x >> 13), c = (int)(item.y & 3u), jb = (int)(item.y >> 2);
                const float2 *payc = pay + (item.x & 8191u);
                const float *payc_y = pay_y + (item.x & 8191u);
                f32x2 m[kKt];
#pragma unroll
                for (int k = 0; k < kKt; ++k) m[k] = 0ull;
                auto add = [&](int src) {
                    const f32x2 w = *reinterpret_cast<const f32x2 *>(payc + src);
                    const float yv = payc_y[src];
                    const f32x2 y2 = pk(yv + yv, yv + yv), ny2 = pk(-(yv + yv), -(yv + yv));
                    f32x2 t0 = pk(1.f, 1.f), t1 = pk(yv, yv);
                    m[0] = fadd2(m[0], w);
                    m[1] = ffma2(w, t1, m[1]);
#pragma unroll
                    for (int k = 2; k < kKt; ++k) {
                        const f32x2 t2 = ffma2((k & 1) ? y2 : ny2, t1, t0);
                        m[k] = ffma2(w, t2, m[k]);
                        t0 = t1; t1 = t2;
                    }
                };
                int i = sub;
                for (; i + 8 < cnt; i += 16) { add(i); add(i + 8); }
                if (i < cnt) add(i);
                // transpose: thread `sub` of the team ends with the team's sum of moment k = sub
                f32x2 *scr64 = reinterpret_cast<f32x2 *>(scr);
#pragma unroll
                for (int k = 0; k < kKt; ++k) scr64[sub * kScrRow + k] = m[k];
                __syncwarp();
                f32x2 hsum = scr64[sub];
#pragma unroll
                for (int r = 1; r < 8; ++r) hsum = fadd2(hsum, scr64[r * kScrRow + sub]);
                __syncwarp();
                float2 h1 = *reinterpret_cast<float2 *>(&hsum);
                if (cnt > 0) {
                    if (sub & 2) { h1.x = -h1.x; h1.y = -h1.y; }
                    atomicAdd(row0 + (size_t)c * cstride + jb, h1);
                }
            }
        }
        // ---- the strays of this pulse: one thread per stray, its eight moments (8 threads per stray made all 8 warps walk
        //      the loop: 5 % of the kernel's instructions) ----
        if (tid < ns) {
            const float4 e = s_stray[buf][tid];
            const int code = __float_as_int(e.w), c = code >> 28, jb = code & 0x0fffffff;
            float2 *row = a.mom + ((size_t)(c * n_pl + pl) * kKt) * a.nb_pad + jb;
            const float y2 = e.z + e.z;
            float t0 = 1.f, t1 = e.z;
            atomicAdd(row, make_float2(e.x, e.y));
            atomicAdd(row + a.nb_pad, make_float2(e.x * t1, e.y * t1));
#pragma unroll
            for (int k = 2; k < kKt; ++k) {
                const float t2 = fmaf(y2, t1, -t0);
                atomicAdd(row + (size_t)k * a.nb_pad, make_float2(e.x * t2, e.y * t2));
                t0 = t1; t1 = t2;
            }
            const int b = jb - (L - 1);
            atomicMin(&s_blo[c], b); atomicMax(&s_bhi[c], b + 1);
        }
        // ---- advance the path of every facet to the next pulse (forward differences) ----
#pragma unroll
        for (int q = 0; q < FPT; ++q) { rho[q] += (unsigned long long)rd1[q]; rd1[q] += rd2[q]; rd2[q] += (long long)rd3[q]; }
        ++ip;
        ns_cur = ns_next;
        if (ns + max(ns - ns_prev, 0) > kStrayCap && ip < hi - lo) { need_sort = true; ip_sort = ip; }   // before the list overflows
        ns_prev = need_sort ? 0 : ns;
        // no barrier here: the next pulse writes the other payload / stray buffers, and this pulse's are rewritten
        // only after the next barrier
    }

    // ---- counters ----
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) my_kept += __shfl_xor_sync(0xffffffffu, my_kept, o);
    if (lane == 0 && my_kept) atomicAdd(&s_kept, my_kept);
    __syncthreads();
    if (tid == 0 && a.counters && s_kept) atomicAdd(a.counters + 0, (unsigned long long)s_kept * C);
    // ---- the band every vector occupies, for K3s (fftconv.cu): outside the pulse loop; a tile with an out-of-window
    //      echo claims the whole row ----
    if (a.band_lo) {
        __syncthreads();                                     // the last pulse's strays have been merged into s_blo / s_bhi
        for (int k = tid; k < (hi - lo) * C; k += NT) {
            const int ip = k / C, c = k - ip * C, v = c * n_pl + (lo + ip - p0);
            // the sorted slices (one more on either side) and the strays, inside the sampling window
            const int blo = max(s_blo[c], -(L - 1)), bhi = min(s_bhi[c], prm.n_samples);
            if (bhi > blo) { atomicMin(a.band_lo + v, blo); atomicMax(a.band_hi + v, bhi); }
        }
    }
}

template <int FPT, int C>
cudaError_t launch_fc(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, int j_first, int n_int,
                      size_t smem, cudaStream_t s)
{
    dim3 grid(prm.k2k_n_tiles, n_int);
    auto go = [&](auto kern) -> cudaError_t {
        // always opt in: static + dynamic shared memory together may pass 48 KB even when the dynamic part does not
        cudaError_t rc = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (rc != cudaSuccess) return rc;
        kern<<<grid, kThreads, smem, s>>>(prm, a, p0, n_pl, j_first);
        return cudaGetLastError();
    };
    if (a.dbg_slice) {                                   // sim_debug_echoes (analytic patterns, static speckle only)
        if (prm.lut_any || a.xi_pulse_stride) return cudaErrorInvalidValue;
        return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, false, false, true>)
                        : go(moments_keyframed_kernel<FPT, C, false, false, false, true>);
    }
    if (prm.lut_any) {
        if (a.xi_pulse_stride)
            return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, true, true, false>) : go(moments_keyframed_kernel<FPT, C, false, true, true, false>);
        return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, false, true, false>) : go(moments_keyframed_kernel<FPT, C, false, false, true, false>);
    }
    if (a.xi_pulse_stride)
        return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, true, false, false>) : go(moments_keyframed_kernel<FPT, C, false, true, false, false>);
    return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, false, false, false>) : go(moments_keyframed_kernel<FPT, C, false, false, false, false>);
}

template <int FPT>
cudaError_t launch_f(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, int j_first, int n_int,
                     size_t smem, cudaStream_t s)
{
    switch (prm.n_channels) {
        case 1: return launch_fc<FPT, 1>(prm, a, p0, n_pl, j_first, n_int, smem, s);
        case 2: return launch_fc<FPT, 2>(prm, a, p0, n_pl, j_first, n_int, smem, s);
        case 3: return launch_fc<FPT, 3>(prm, a, p0, n_pl, j_first, n_int, smem, s);
        case 4: return launch_fc<FPT, 4>(prm, a, p0, n_pl, j_first, n_int, smem, s);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

// slice index in 12 bits, slot rank in 12 bits, slot position in 13 bits, shared memory of one CTA
bool moments_keyframed_fits(const DevParams &prm, int span_cap)
{
    return span_cap < 4096 && prm.k2k_cap <= 1024 && (prm.k2k_cap <= kThreads || prm.k2k_cap == 3 * kThreads) &&
           prm.n_channels <= kMaxKeyChannels && prm.n_channels * prm.k2k_cap + 2 <= 8191 &&
           moments_keyframed_smem_bytes(prm, span_cap) <= 200 * 1024;
}

size_t moments_keyframed_smem_bytes(const DevParams &prm, int span_cap)
{
    const size_t C = prm.n_channels;
    return (size_t)2 * (C * prm.k2k_cap + 2) * 12 + C * prm.k2k_cap * 4 + (size_t)hist_words((int)C, span_cap) * 4 +
           (size_t)(kThreads / 8) * kScrTeam * sizeof(float2) + (size_t)item_words((int)C, span_cap) * sizeof(uint2) +
           (size_t)6 * kThreads * sizeof(float2);
}

cudaError_t launch_moments_keyframed(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, cudaStream_t s)
{
    const int H = a.surf.H, P = a.surf.n_pulses_total;
    if (H <= 1 || H + 1 > kMaxKeyPulses || prm.n_channels > kMaxKeyChannels || !prm.series_channels ||
        !moments_keyframed_fits(prm, a.span_cap))
        return cudaErrorInvalidValue;
    const int n_keys = (P - 1 + H - 1) / H + 1;
    const int j_first = min(p0 / H, n_keys - 2), j_last = min((p0 + n_pl - 1) / H, n_keys - 2);
    const int n_int = j_last - j_first + 1;
    const size_t smem = moments_keyframed_smem_bytes(prm, a.span_cap);
    if (prm.k2k_cap <= kThreads) return launch_f<1>(prm, a, p0, n_pl, j_first, n_int, smem, s);
    return launch_f<3>(prm, a, p0, n_pl, j_first, n_int, smem, s);
}

}  // namespace heeps
