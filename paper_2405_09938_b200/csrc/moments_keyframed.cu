// K2k -- geometry, gains, amplitude, cull and range-slice moments with the GEOMETRY evaluated exactly only
// at the kinematics keyframes (SURVEY.md §8(a) A2..A6 moment form).
//
// moments.cu evaluates the fp64 antenna legs and the sinc patterns of every facet at every pulse: 1156
// instructions per facet-pulse, issue-bound (profiles/r1_v4).  But over one keyframe interval (H pulses, a few
// milliseconds) everything a facet-echo needs is a smooth function of time:
//
//   R(t)   = r_t + r_r,ref  bistatic path to the un-offset phase centre: cubic HERMITE from the exact values and
//            time derivatives at the two keyframes,  dR/dt = u_t.(v_f - V_tx) + u_r.(v_f - V_rx)  with the facet
//            velocity v_f = (current + dD_h/dt, dz/dt) from K1's rate rows.  Error <= h^4 max|R''''| / 384:
//            platform term 3 V^4/r^3 ~ 0.02 m/s^4 -> 4e-13 m at h = 9.4 ms; wave term = K1's own bound (2e-9 m).
//   d_c(t) = r_r,c - r_r,ref  (receive phase centre c, |o_c| <= 1e-4 r) = o_c a(t) + o_c^2 b, a = -(d.v^)/r linear
//            in t, b = (1 - a^2)/(2 r); fp32 (|d_c| < 1 m).
//   P(t)   = G_t G_r,ref      quadratic through t0, t_mid, t1 with the sinc arguments at t_mid taken as the mean of
//            the end values (they are linear in t to ~1e-7); G_r,c = G_r,ref + o_c dG/do with dG/do by one
//            finite difference at t_mid.  |a_f|(t) (tilt modulation) quadratic the same way.
//
// sim_create verifies these three interpolants against the exact geometry on a 3 x 3 lattice of scene points
// at EVERY pulse (host, long double) and falls back to moments.cu when any bound fails (sim_api.cu
// geometry_keyframes_ok): non-smooth state vectors never reach this kernel.
//
// One CTA = one spatial tile x one keyframe interval.  A thread owns FPT facets, holds their interpolants in
// registers (18 words per facet) and loops over the interval's pulses.  The tile's facet-echoes (all C channels) are
// ordered by range slice ONCE per interval -- counting sort at its middle pulse: shared-memory histogram by integer
// ATOMS, scan, slot = first position of the slice + rank -- because over a few milliseconds a facet changes slice only
// when its sub-slice position crosses 0 or 1 (a percent or two of the echoes per pulse).  Per pulse: (A) slice,
// sub-slice position and complex weight of every facet-echo; an echo found in its sorted slice writes its weight into
// its slot, one found elsewhere ("stray") leaves a zero there and goes to a short shared-memory list; one barrier;
// (C) 8 threads per occupied slice (one work list over all channels) sum the Kt Chebyshev moments of the slice's
// contiguous slots (packed FFMA2), transpose through shared memory, one RED.ADD.F32x2 per (slice, k); the strays are
// worked off with global atomics, thread t taking moment t & 7 of stray t >> 3.  A pulse whose strays would not fit
// the list sorts the tile again (and is redone if they did not fit).  Payload and stray list are double-buffered.
//
// Bound: issue slots (FP32 + FP64 mix); HBM/L2: four surface rows per facet and INTERVAL, the maps once.
#include "kernels.cuh"
#include "geometry_common.cuh"

namespace heeps {

namespace {

constexpr int kThreads = 256;
constexpr int kKt = kMomentOrder;
static_assert(kKt == 8, "the reduce-scatter below is written for 8 moments / 8 threads per slice");

struct __align__(16) KeyPulse {          // per pulse of the interval (shared memory)
    double sd;                           // (t - t0) / h
    float u0, u1;                        // s (1-s)^2, -s^2 (1-s): weights of the Hermite cubic's bend (see R below)
    double r0;                           // c0 t0[p]
    float s, pad0;                       // (t - t0) / h
    int32_t base[kMaxKeyChannels];       // first slice of the tile's shared-memory window, per channel
};

// Exact state of one facet at one keyframe pulse.
template <int C>
struct KeyEval {
    double R, Rd;                        // path to the un-offset phase centre and its time derivative
    float xat, xet, xar, xer;            // sinc arguments: Tx azimuth / elevation, Rx (un-offset) azimuth / elevation
    float xao, xeo;                      // Rx arguments at the finite-difference offset o_fd
    float la, lb;                        // r_r,c - r_r,ref = o_c la + o_c^2 lb  (series in o_c / r)
    double uat, uet, uar, uer, uao, ueo; // the same six as direction cosines (tabulated patterns: grid coordinates in fp64)
};

template <int C>
__device__ __forceinline__ KeyEval<C> key_eval(const DevParams &prm, const PulseConst &pc, const double pos[3],
                                               const double vel[3], double o_fd)
{
    KeyEval<C> o;
    const LegParts lt = leg_parts(pos, pc.tx_pos, pc.tx_a, pc.tx_e);
    const LegParts lr = leg_parts(pos, pc.rx_ref, pc.rx_a, pc.rx_e);
    o.R = lt.r + lr.r;
    const double at = fma(lt.dx, vel[0] - pc.tx_vel[0], fma(lt.dy, vel[1] - pc.tx_vel[1], lt.dz * (vel[2] - pc.tx_vel[2])));
    const double ar = fma(lr.dx, vel[0] - pc.rx_vel[0], fma(lr.dy, vel[1] - pc.rx_vel[1], lr.dz * (vel[2] - pc.rx_vel[2])));
    o.Rd = fma(at, lt.inv, ar * lr.inv);
    o.xat = (float)(prm.ap_tx_a * (lt.da * lt.inv)); o.xet = (float)(prm.ap_tx_e * (lt.de * lt.inv));
    o.xar = (float)(prm.ap_rx_a * (lr.da * lr.inv)); o.xer = (float)(prm.ap_rx_e * (lr.de * lr.inv));
    o.uat = lt.da * lt.inv; o.uet = lt.de * lt.inv; o.uar = lr.da * lr.inv; o.uer = lr.de * lr.inv;
    const double dv = fma(lr.dx, pc.rx_vhat[0], fma(lr.dy, pc.rx_vhat[1], lr.dz * pc.rx_vhat[2]));
    {
        double r_c, inv_c, da_c, de_c;
        channel_leg_series(lr, dv, o_fd, pc.rx_va, pc.rx_ve, r_c, inv_c, da_c, de_c);
        o.xao = (float)(prm.ap_rx_a * (da_c * inv_c)); o.xeo = (float)(prm.ap_rx_e * (de_c * inv_c));
        o.uao = da_c * inv_c; o.ueo = de_c * inv_c;
    }
    // r_c - r = r (dl/2 - dl^2/8 + ...), dl = (o^2 - 2 o d.v^)/r^2  (geometry_common.cuh)
    //         = -o (d.v^)/r + o^2 (1 - (d.v^/r)^2)/(2 r) + O(o^3/r^2)
    const double cv = dv * lr.inv;
    o.la = (float)(-cv);
    o.lb = (float)(0.5 * lr.inv * fma(-cv, cv, 1.0));
    return o;
}

constexpr int kStrayCap = 96;             // stray echoes of one pulse held in shared memory (more: the tile is sorted again)
constexpr int kScrRow = 9;                // float2 per thread row of the transposition scratch (8 moments + 1 pad)
constexpr int kScrTeam = 8 * kScrRow;     // float2 per 8-thread team
__host__ __device__ constexpr int hist_words(int C, int span) { return (2 * C * (span + 1) + 1) & ~1; }

// Packed f32x2 arithmetic on 64-bit registers (FFMA2 / FADD2): the operands stay register pairs from the
// shared-memory load to the transposition store, no pack / unpack moves in the moment loop.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float x, float y)
{
    f32x2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(x), "f"(y));
    return d;
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
__device__ __forceinline__ float2 gain_at(const DevParams &prm, int k, double ua, double ue)
{
    if (prm.lut[k].tab) return lut_gain(prm.lut[k], ua, ue);
    const double apa = k ? prm.ap_rx_a : prm.ap_tx_a, ape = k ? prm.ap_rx_e : prm.ap_tx_e;
    return make_float2(pattern_x((float)(apa * ua), (float)(ape * ue)), 0.f);
}

template <int FPT, int C, bool kTilt, bool kSpeckleT, bool kLut>
__global__ void __launch_bounds__(kThreads, 2)
moments_keyframed_kernel(DevParams prm, MomentArgs a, int p0, int n_pl, int j_first)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ PulseConst pc2[2];
    __shared__ KeyPulse s_kp[kMaxKeyPulses];
    __shared__ double s_rc[2][kMaxKeyChannels];          // path length of the tile centre at the two keyframes
    __shared__ unsigned long long s_samples;
    __shared__ int s_kept;
    __shared__ int s_rng[kMaxKeyChannels][2];
    __shared__ float4 s_stray[2][kStrayCap];                     // echoes that have left their sorted slice: (w, y, row index)
    __shared__ int s_nstray[3];
    __shared__ int s_blo[kMaxKeyChannels], s_bhi[kMaxKeyChannels];   // slices this tile touches during the interval

    const int span = a.span_cap, hstride = span + 1;
    const int cap = prm.tile_cap;
    // [2][C][cap] float2 weight | [2][C][cap] float y | [2][C][cap] u16 index list | [2][C][span + 1] int histogram |
    // [kThreads / 8][kScrTeam] float2 transposition scratch of stage C (8-byte aligned: hist is padded)
    float2 *payload = reinterpret_cast<float2 *>(smem_raw);
    float *payload_y = reinterpret_cast<float *>(smem_raw + (size_t)2 * C * cap * 8);
    unsigned short *idx = reinterpret_cast<unsigned short *>(smem_raw + (size_t)2 * C * cap * 12);
    int *hist = reinterpret_cast<int *>(smem_raw + (size_t)2 * C * cap * 14);
    float2 *scratch = reinterpret_cast<float2 *>(smem_raw + (size_t)2 * C * cap * 14 + (size_t)hist_words(C, span) * 4);

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
        for (int k = tid; k < (int)(sizeof(PulseConst) / sizeof(double)); k += kThreads) { d0[k] = s0[k]; d1[k] = s1[k]; }
    }
    if (tid == 0) { s_samples = 0ull; s_kept = 0; s_nstray[0] = s_nstray[1] = s_nstray[2] = 0; }
    if (tid < kMaxKeyChannels) { s_blo[tid] = 0x7fffffff; s_bhi[tid] = (int)0x80000000; }
    for (int k = tid; k < C * hstride; k += kThreads) hist[k] = 0;
    __syncthreads();

    const int ts = prm.tile, lts = 31 - __clz(ts);
    const int ti0 = (tile % prm.tiles_x) * ts, tj0 = (tile / prm.tiles_x) * ts;
    if (tid < 2 * C) {
        // tile centre (rest, flat) at the two keyframes: positions the slice window of every pulse between
        const int e = tid / C, c = tid - e * C;
        const PulseConst &pc = pc2[e];
        const double ic = ti0 + 0.5 * (min(ts, prm.nx - ti0) - 1), jc = tj0 + 0.5 * (min(ts, prm.ny - tj0) - 1);
        const double x = prm.cx + (ic - 0.5 * (prm.nx - 1)) * prm.spacing;
        const double y = prm.cy + (jc - 0.5 * (prm.ny - 1)) * prm.spacing;
        const double ax = x - pc.tx_pos[0], ay = y - pc.tx_pos[1], az = prm.cz - pc.tx_pos[2];
        const double bx = x - pc.rx_pos[c][0], by = y - pc.rx_pos[c][1], bz = prm.cz - pc.rx_pos[c][2];
        s_rc[e][c] = sqrt(ax * ax + ay * ay + az * az) + sqrt(bx * bx + by * by + bz * bz);
    }
    __syncthreads();
    for (int ip = tid; ip < hi - lo; ip += kThreads) {
        const int p = lo + ip;
        const double t0 = pc2[0].t, t1 = pc2[1].t, t = a.pulses[p].t;
        const double h = t1 - t0;
        const double s = (h != 0.0) ? (t - t0) / h : 0.0;
        const double s2 = s * s, s3 = s2 * s;
        KeyPulse kp;
        kp.sd = s;
        kp.u0 = (float)(s3 - 2.0 * s2 + s);
        kp.u1 = (float)(s3 - s2);
        kp.r0 = a.pulses[p].r0;
        kp.s = (float)s; kp.pad0 = 0.f;
#pragma unroll
        for (int c = 0; c < kMaxKeyChannels; ++c) {
            int base = 0;
            if (c < C) {
                const double rc = fma(s, s_rc[1][c] - s_rc[0][c], s_rc[0][c]);
                double bc = ceil((rc - kp.r0) * prm.fs_over_c0 - prm.half_len) - 0.5 * span;
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

    // Hermite cubic of the path length as chord + bend:  R(s) = R0 + s D + u0(s) ra + u1(s) rb,  D = R1 - R0,
    // ra = h R0' - D, rb = h R1' - D.  The bend is millimetres (h^2 R''/8), so ra, rb are fp32.
    double R0[FPT], RD[FPT];
    float ra[FPT], rb[FPT];
    float la0[FPT], dla[FPT];                            // r_r,c - r_r,ref = o_c (la0 + s dla) + o_c^2 lb
    float lb_sum = 0.f;                                  // lb varies by 1e-4 relative over a tile: one value per thread
    int lb_n = 0;
    float pq0[FPT], pqa[FPT], pqb[FPT], bq[FPT];         // P(s) = pq0 + s (pqa + s pqb); bq = G_t dG_r/do
    constexpr int FL = kLut ? FPT : 1;                   // tabulated patterns: P and bq are complex, these are the imaginary parts
    float qi0[FL], qia[FL], qib[FL], bqi[FL];
    float am0[FPT], ama[FPT], amb[FPT];                  // |a_f|(s), quadratic when tilt-modulated
    uint32_t xarg[FPT];
    bool valid[FPT];
#pragma unroll
    for (int q = 0; q < FPT; ++q) {
        const int k = q * kThreads + tid;
        const int li = k & (ts - 1), lj = k >> lts;
        const int i = ti0 + li, jj = tj0 + lj;
        valid[q] = (k < ts * ts && i < prm.nx && jj < prm.ny);
        R0[q] = RD[q] = 0.0; ra[q] = rb[q] = 0.f;
        pq0[q] = pqa[q] = pqb[q] = bq[q] = 0.f; am0[q] = ama[q] = amb[q] = 0.f; xarg[q] = 0u;
        la0[q] = dla[q] = 0.f;
        if (kLut) qi0[q] = qia[q] = qib[q] = bqi[q] = 0.f;
        if (!valid[q]) continue;
        const size_t f = (size_t)jj * prm.nx + i;
        const double xb = prm.cx + ((double)i - 0.5 * (prm.nx - 1)) * prm.spacing;
        const double yb = prm.cy + ((double)jj - 0.5 * (prm.ny - 1)) * prm.spacing;
        double cux = prm.cur_ux, cuy = prm.cur_uy;
        if (a.current) { const float2 cv = __ldg(a.current + f); cux = cv.x; cuy = cv.y; }
        KeyEval<C> ev[2];
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
            ev[e] = key_eval<C>(prm, pc, pos, vel, o_fd);
        }
        {
            const double hh = pc2[1].t - pc2[0].t, D = ev[1].R - ev[0].R;
            R0[q] = ev[0].R; RD[q] = D;
            ra[q] = (float)fma(hh, ev[0].Rd, -D); rb[q] = (float)fma(hh, ev[1].Rd, -D);
        }
        la0[q] = ev[0].la; dla[q] = ev[1].la - ev[0].la;
        lb_sum += 0.5f * (ev[0].lb + ev[1].lb); ++lb_n;
        // gains at s = 0, 1/2, 1 (sinc arguments at the midpoint = mean of the end values)
        if (kLut) {
            const float2 P0 = cmulf(gain_at(prm, 0, ev[0].uat, ev[0].uet), gain_at(prm, 1, ev[0].uar, ev[0].uer));
            const float2 P1 = cmulf(gain_at(prm, 0, ev[1].uat, ev[1].uet), gain_at(prm, 1, ev[1].uar, ev[1].uer));
            const float2 gtm = gain_at(prm, 0, 0.5 * (ev[0].uat + ev[1].uat), 0.5 * (ev[0].uet + ev[1].uet));
            const float2 grm = gain_at(prm, 1, 0.5 * (ev[0].uar + ev[1].uar), 0.5 * (ev[0].uer + ev[1].uer));
            const float2 gom = gain_at(prm, 1, 0.5 * (ev[0].uao + ev[1].uao), 0.5 * (ev[0].ueo + ev[1].ueo));
            const float2 Pm = cmulf(gtm, grm);
            const float2 dq = cmulf(gtm, make_float2((gom.x - grm.x) * inv_ofd, (gom.y - grm.y) * inv_ofd));
            pq0[q] = P0.x; pqa[q] = -3.f * P0.x + 4.f * Pm.x - P1.x; pqb[q] = 2.f * P0.x - 4.f * Pm.x + 2.f * P1.x;
            qi0[q] = P0.y; qia[q] = -3.f * P0.y + 4.f * Pm.y - P1.y; qib[q] = 2.f * P0.y - 4.f * Pm.y + 2.f * P1.y;
            bq[q] = dq.x; bqi[q] = dq.y;
        } else {
        const float gt0 = pattern_x(ev[0].xat, ev[0].xet), gr0 = pattern_x(ev[0].xar, ev[0].xer);
        const float gt1 = pattern_x(ev[1].xat, ev[1].xet), gr1 = pattern_x(ev[1].xar, ev[1].xer);
        const float gtm = pattern_x(0.5f * (ev[0].xat + ev[1].xat), 0.5f * (ev[0].xet + ev[1].xet));
        const float grm = pattern_x(0.5f * (ev[0].xar + ev[1].xar), 0.5f * (ev[0].xer + ev[1].xer));
        const float gom = pattern_x(0.5f * (ev[0].xao + ev[1].xao), 0.5f * (ev[0].xeo + ev[1].xeo));
        const float P0 = gt0 * gr0, Pm = gtm * grm, P1 = gt1 * gr1;
        pq0[q] = P0; pqa[q] = -3.f * P0 + 4.f * Pm - P1; pqb[q] = 2.f * P0 - 4.f * Pm + 2.f * P1;
        bq[q] = gtm * (gom - grm) * inv_ofd;
        }
        // amplitude (O8): sqrt(sigma0 tilt d^2) |xi|
        const float sig = a.sigma0 ? __ldg(a.sigma0 + f) : (float)prm.sigma0_uniform;
        // static speckle: |xi| and arg xi are constants of the facet; time-dependent speckle (speckle.cu): per pulse
        float xmag = 1.f;
        if (!kSpeckleT) { const uint2 xp = __ldg(a.xi_polar + f); xmag = __uint_as_float(xp.x); xarg[q] = xp.y; }
        if (kTilt) {
            const float2 sl0 = a.surf.slope[row0 + f], sl1 = a.surf.slope[row1 + f];
            const float smx = 0.5f * (sl0.x + sl1.x), smy = 0.5f * (sl0.y + sl1.y);   // slopes are linear between keyframes
            const float lx = (float)prm.look_x, ly = (float)prm.look_y;
            const float A0 = sqrtf(sig * fmaxf(1.f + 2.f * (sl0.x * lx + sl0.y * ly), 0.f) * area) * xmag;
            const float Am = sqrtf(sig * fmaxf(1.f + 2.f * (smx * lx + smy * ly), 0.f) * area) * xmag;
            const float A1 = sqrtf(sig * fmaxf(1.f + 2.f * (sl1.x * lx + sl1.y * ly), 0.f) * area) * xmag;
            am0[q] = A0; ama[q] = -3.f * A0 + 4.f * Am - A1; amb[q] = 2.f * A0 - 4.f * Am + 2.f * A1;
        } else {
            am0[q] = sqrtf(sig * area) * xmag;
        }
    }
    __syncthreads();                                     // s_kp complete

    // phase of a facet-echo in 2^-32 turns: -dR/lambda + kappa eps^2 (+ speckle argument, + 1/2 if the gain is negative)
    const double il32 = prm.inv_lambda * 4294967296.0;
    const float kappa32 = (float)(prm.kappa * 4294967296.0);
    const int L = a.replica;
    const unsigned win_hi = (unsigned)(prm.n_samples + L - 1);
    float och[C];
#pragma unroll
    for (int c = 0; c < C; ++c) och[c] = (float)pc2[0].ch_off[c];
    const float lbt = lb_n ? lb_sum / (float)lb_n : 0.f;
    unsigned long long my_samples = 0;
    int my_kept = 0;
    const int sub = tid & 7, team = tid >> 3, warp = tid >> 5;
    float2 *scr = scratch + team * kScrTeam;

    // ---- The facet-echoes of the tile are ordered by range slice ONCE (counting sort at the interval's middle pulse:
    //      histogram by integer ATOMS, scan, slot = first position of the slice + rank), not at every pulse: over the
    //      few milliseconds of an interval a facet's slice changes only when its sub-slice position crosses 0 or 1
    //      (the window follows the scene: a percent or two of the echoes per pulse).  At every pulse an echo found in
    //      its sorted slice writes its weight into its slot; one found elsewhere ("stray") leaves a zero there and goes
    //      to a short shared-memory list that the CTA works off with global atomics.  A pulse with more strays than the
    //      list holds sorts the tile again at that pulse and is redone.  Stage C reads each slice's slots
    //      contiguously: no per-pulse histogram, scan or index list; one barrier per pulse. ----
    uint32_t *slots = reinterpret_cast<uint32_t *>(idx);           // [C][cap]: slice << 12 | slot, or ~0u (never in the list)
    int *hs = hist;                                                  // [C][span + 1] first slot of each slice
    int bref[C];                                                     // first slice of the tile's window at the sorting pulse
    // Sorted at the middle pulse of the interval the strays at its ends are half as many as when sorted at the first;
    // a tile far from the scene centre drifts too fast for that (expected strays at the first pulse = half the
    // interval's pulses x the drift of the tile centre against the sampling window, in slices per pulse, x its echoes):
    // it is sorted at the first pulse, and again whenever the next pulse's strays (this pulse's plus their growth)
    // would not fit the list.
    int ip_sort = (hi - lo) / 2;
    {
        const double drift = fabs((s_rc[1][0] - s_rc[0][0]) - (a.pulses[k1].r0 - a.pulses[k0].r0)) * prm.fs_over_c0 /
                             (double)max(k1 - k0, 1);
        if (drift * (double)(ts * ts * C) * 0.5 * (double)(hi - lo) > 0.9 * kStrayCap) ip_sort = 0;
    }
    bool need_sort = true;
    int ns_prev = 0;                                                 // strays of the previous pulse (0 after a sort)

    for (int ip = 0; ip < hi - lo;) {
        if (need_sort) {
            need_sort = false;
            const KeyPulse &kp = s_kp[ip_sort];
            __syncthreads();                                         // nobody reads the old histogram / slots any more
            for (int k = tid; k < C * hstride; k += kThreads) hs[k] = 0;
            if (tid == 0) s_nstray[ip % 3] = 0;
            __syncthreads();
#pragma unroll
            for (int c = 0; c < C; ++c) bref[c] = kp.base[c];
            int pr[FPT][C];
#pragma unroll
            for (int q = 0; q < FPT; ++q) {
                const double dRref = fma(kp.sd, RD[q], R0[q]) + (double)fmaf(kp.u0, ra[q], kp.u1 * rb[q]) - kp.r0;
                const float la = fmaf(kp.s, dla[q], la0[q]);
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    const float dl = och[c] * fmaf(och[c], lbt, la);
                    const int rel = __double2int_ru(fma(dRref + (double)dl, prm.fs_over_c0, -prm.half_len)) - bref[c];
                    pr[q][c] = -1;
                    if (valid[q] && (unsigned)rel < (unsigned)span)
                        pr[q][c] = (rel << 12) | atomicAdd(&hs[c * hstride + rel + 1], 1);
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
#pragma unroll
            for (int q = 0; q < FPT; ++q)
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    const int v = pr[q][c];
                    if (FPT > 1 || q * kThreads + tid < cap)         // (FPT = 1: the tile may be smaller than the CTA)
                        slots[c * cap + q * kThreads + tid] =
                            (v >= 0) ? (uint32_t)((v & ~4095) | (hs[c * hstride + (v >> 12)] + (v & 4095))) : 0xffffffffu;
                }
            // a thread reads only its own slots; the scan results are read after the barrier of stage A
        }
        const int buf = ip & 1;
        const int pl = lo + ip - p0;
        const KeyPulse &kp = s_kp[ip];
        float2 *pay = payload + (size_t)buf * C * cap;
        float *pay_y = payload_y + (size_t)buf * C * cap;
        const float s = kp.s;
        int *n_stray = &s_nstray[ip % 3];
        if (tid == 0) s_nstray[(ip + 1) % 3] = 0;            // last read two pulses ago, next written after this pulse's barrier
        int kept_p = 0;
        unsigned samples_p = 0;

        // ---- A: slice, sub-slice position, complex weight of every facet-echo, written to the echo's slot.
        //      Straight-line code for all FPT x C echoes of the thread (predicated stores), so that the
        //      independent chains interleave; only a stray echo branches.
#pragma unroll
        for (int q = 0; q < FPT; ++q) {
            const float Pv = fmaf(s, fmaf(s, pqb[q], pqa[q]), pq0[q]);
            const float Pi = kLut ? fmaf(s, fmaf(s, qib[kLut ? q : 0], qia[kLut ? q : 0]), qi0[kLut ? q : 0]) : 0.f;
            const bool keep = valid[q] && !(kLut ? (fmaf(Pv, Pv, Pi * Pi) < prm.cull_thr * prm.cull_thr)
                                                 : (fabsf(Pv) < prm.cull_thr));     // O7 (G6)
            kept_p += keep ? 1 : 0;
            float am = kTilt ? fmaf(s, fmaf(s, amb[q], ama[q]), am0[q]) : am0[q];
            uint32_t xa = xarg[q];
            if (kSpeckleT && valid[q]) {                  // time-dependent speckle: s_f(t_p) of this pulse (eq. (7), (10))
                const int kk = q * kThreads + tid;
                const uint2 xp = __ldg(a.xi_polar + (size_t)pl * a.xi_pulse_stride +
                                       (size_t)(tj0 + (kk >> lts)) * prm.nx + (ti0 + (kk & (ts - 1))));
                am *= __uint_as_float(xp.x); xa = xp.y;
            }
            const double R = fma(kp.sd, RD[q], R0[q]) + (double)fmaf(kp.u0, ra[q], kp.u1 * rb[q]);
            const double dRref = R - kp.r0;
            const float la = fmaf(s, dla[q], la0[q]);
            const int k = q * kThreads + tid;
#pragma unroll
            for (int c = 0; c < C; ++c) {
                const float dl = och[c] * fmaf(och[c], lbt, la);
                const double dR = dRref + (double)dl;
                const double nu = fma(dR, prm.fs_over_c0, -prm.half_len);
                const int b = __double2int_ru(nu);                                // ceil, saturating
                const bool inwin = keep && ((unsigned)b + (unsigned)(L - 1) < win_hi);   // window meets [0, Ns)
                const float eps = (float)((double)b - nu);                        // [0, 1)
                const float g = fmaf(och[c], bq[q], Pv);
                const uint32_t ph = (uint32_t)(unsigned long long)__double2ll_rn(
                                        fma(-dR, il32, (double)(kappa32 * eps * eps))) +
                                    xa + ((g < 0.f && !kLut) ? 0x80000000u : 0u);
                float sn, cs;
                __sincosf((float)(int32_t)ph * 1.4629180792671596e-9f, &sn, &cs);   // 2 pi / 2^32
                const float mag = fabsf(g) * am;
                float wr = mag * cs, wi = mag * sn;                        // complex weight of the facet-echo
                if (kLut) {                                                // complex gain times the phasor
                    const float gi = fmaf(och[c], bqi[kLut ? q : 0], Pi);
                    wr = am * fmaf(g, cs, -gi * sn); wi = am * fmaf(g, sn, gi * cs);
                }
                const float yv = fmaf(2.f, eps, -1.f);
                const uint32_t slot = (FPT > 1 || k < cap) ? slots[c * cap + k] : 0xffffffffu;
                const int rel = b - bref[c];
                const bool here = inwin && ((uint32_t)rel == (slot >> 12));       // in its sorted slice
                if (slot != 0xffffffffu) {
                    const int pos = c * cap + (int)(slot & 4095u);
                    pay[pos] = here ? make_float2(wr, wi) : make_float2(0.f, 0.f);
                    pay_y[pos] = here ? yv : 0.f;
                }
                if (inwin) samples_p += (unsigned)(min(b + L, prm.n_samples) - max(b, 0));
                if (inwin && !here) {                                      // stray: left its sorted slice, or never had one
                    const int t = atomicAdd(n_stray, 1);
                    if (t < kStrayCap) s_stray[buf][t] = make_float4(wr, wi, yv, __int_as_float((c << 28) | (b + L - 1)));
                }
            }
        }
        __syncthreads();
        const int ns = *n_stray;
        if (ns > kStrayCap) {                                // too many have moved on: sort the tile at this pulse, redo it
            need_sort = true; ip_sort = ip;
            continue;
        }
        my_kept += kept_p; my_samples += samples_p;

        // ---- C: 8 threads per slice: Chebyshev moments over the slice's slots, transpose through shared memory, one
        //      RED per (slice, k).  The recurrence runs on a_k = sigma_k T_k, sigma = + + - - + + - -, which needs no
        //      negation: a_{k+1} = -+ 2y a_k + a_{k-1} (minus for odd k); sigma_k is applied to the slice sum.
        //      Work items = the occupied slices of all C channels laid end to end.
        {
            int pre[C + 1];                                                // first item of channel c
            pre[0] = 0;
#pragma unroll
            for (int c = 0; c < C; ++c) pre[c + 1] = pre[c] + max(s_rng[c][1] - s_rng[c][0], 0);
            const int total = pre[C];
            for (int it0 = 0; it0 < total; it0 += kThreads / 8) {
                if (it0 + warp * 4 >= total) break;                        // warp-uniform
                const int it = it0 + team;
                int c = 0;
#pragma unroll
                for (int cc = 1; cc < C; ++cc) c = (it >= pre[cc]) ? cc : c;
                int pc0 = 0, bc = bref[0];
#pragma unroll
                for (int cc = 1; cc < C; ++cc) { pc0 = (c == cc) ? pre[cc] : pc0; bc = (c == cc) ? bref[cc] : bc; }
                const int sidx = s_rng[c][0] + (it - pc0);
                const int *hc = hs + c * hstride;
                int first = 0, cnt = 0;
                if (it < total) { first = hc[sidx]; cnt = hc[sidx + 1] - first; }
                const int b = bc + sidx;
                if ((unsigned)(b + L - 1) >= win_hi) cnt = 0;              // a slice outside the sampling window holds zeros only
                const float2 *payc = pay + c * cap + first;
                const float *payc_y = pay_y + c * cap + first;
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
                    float2 *row = a.mom + ((size_t)(c * n_pl + pl) * kKt + sub) * a.nb_pad;
                    atomicAdd(row + (b + L - 1), h1);
                }
            }
        }
        // ---- the strays of this pulse: thread t takes moment t & 7 of stray t >> 3 ----
        for (int t = tid; t < ns * kKt; t += kThreads) {
            const float4 e = s_stray[buf][t >> 3];
            const int k = t & 7, code = __float_as_int(e.w), c = code >> 28, jb = code & 0x0fffffff;
            float t0 = 1.f, t1 = e.z;
            for (int kk = 1; kk < k; ++kk) { const float t2 = 2.f * e.z * t1 - t0; t0 = t1; t1 = t2; }
            const float tk = k ? t1 : 1.f;
            atomicAdd(a.mom + ((size_t)(c * n_pl + pl) * kKt + k) * a.nb_pad + jb, make_float2(e.x * tk, e.y * tk));
            if (k == 0) { const int b = jb - (L - 1); atomicMin(&s_blo[c], b); atomicMax(&s_bhi[c], b + 1); }
        }
        ++ip;
        if (ns + max(ns - ns_prev, 0) > kStrayCap && ip < hi - lo) { need_sort = true; ip_sort = ip; }   // before the list overflows
        ns_prev = need_sort ? 0 : ns;
        // no barrier here: the next pulse writes the other payload / stray buffers, and this pulse's are rewritten
        // only after the next barrier
    }

    // ---- counters ----
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_samples += __shfl_xor_sync(0xffffffffu, my_samples, o);
        my_kept += __shfl_xor_sync(0xffffffffu, my_kept, o);
    }
    if (lane == 0) {
        if (my_samples) atomicAdd(&s_samples, my_samples);
        if (my_kept) atomicAdd(&s_kept, my_kept);
    }
    __syncthreads();
    if (tid == 0 && a.counters) {
        if (s_kept) atomicAdd(a.counters + 0, (unsigned long long)s_kept * C);
        if (s_samples) atomicAdd(a.counters + 1, s_samples);
    }
    // ---- the band every vector occupies, for K3s (fftconv.cu): outside the pulse loop, whose code must stay as it is
    //      (two atomics inside it cost 4 % of the kernel); a tile with an out-of-window echo claims the whole row ----
    if (a.band_lo) {
        __syncthreads();                                     // the last pulse's strays have been merged into s_blo / s_bhi
        for (int k = tid; k < (hi - lo) * C; k += kThreads) {
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
    dim3 grid(prm.n_tiles, n_int);
    auto go = [&](auto kern) -> cudaError_t {
        // always opt in: static + dynamic shared memory together may pass 48 KB even when the dynamic part does not
        cudaError_t rc = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (rc != cudaSuccess) return rc;
        kern<<<grid, kThreads, smem, s>>>(prm, a, p0, n_pl, j_first);
        return cudaGetLastError();
    };
    if (prm.lut_any) {
        if (a.xi_pulse_stride)
            return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, true, true>) : go(moments_keyframed_kernel<FPT, C, false, true, true>);
        return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, false, true>) : go(moments_keyframed_kernel<FPT, C, false, false, true>);
    }
    if (a.xi_pulse_stride)
        return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, true, false>) : go(moments_keyframed_kernel<FPT, C, false, true, false>);
    return prm.tilt ? go(moments_keyframed_kernel<FPT, C, true, false, false>) : go(moments_keyframed_kernel<FPT, C, false, false, false>);
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

size_t moments_keyframed_smem_bytes(const DevParams &prm, int span_cap)
{
    const size_t C = prm.n_channels;
    return (size_t)2 * C * prm.tile_cap * 14 + (size_t)hist_words((int)C, span_cap) * 4 +
           (size_t)(kThreads / 8) * kScrTeam * sizeof(float2);
}

cudaError_t launch_moments_keyframed(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, cudaStream_t s)
{
    const int H = a.surf.H, P = a.surf.n_pulses_total;
    if (H <= 1 || H + 1 > kMaxKeyPulses || prm.n_channels > kMaxKeyChannels || !prm.series_channels ||
        a.span_cap >= (1 << 19) || prm.tile_cap > 4096)
        return cudaErrorInvalidValue;
    const int n_keys = (P - 1 + H - 1) / H + 1;
    const int j_first = min(p0 / H, n_keys - 2), j_last = min((p0 + n_pl - 1) / H, n_keys - 2);
    const int n_int = j_last - j_first + 1;
    const size_t smem = moments_keyframed_smem_bytes(prm, a.span_cap);
    if (prm.tile_cap <= kThreads) return launch_f<1>(prm, a, p0, n_pl, j_first, n_int, smem, s);
    if (prm.tile_cap <= 4 * kThreads) return launch_f<4>(prm, a, p0, n_pl, j_first, n_int, smem, s);
    return cudaErrorInvalidValue;
}

}  // namespace heeps
