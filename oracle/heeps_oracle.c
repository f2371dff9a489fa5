/*
 * heeps_oracle.c -- plain, slow, fp64 CPU oracle of the raw-data generator hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2405_09938_b200/) may
 * include, link, import or execute this file; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs call it.  It shares no code, header,
 * table or constant generator with the CUDA path.
 *
 * What it computes (BASELINE.json north_star; scalar form of PAPER.md eq. (3) line 91 and
 * eq. (16), with the range-slice sum of eq. (17) lines 204-209 written out as
 * explicit chirp replicas -- the paper convolves the sliced impulse response with the
 * waveform afterwards):
 *
 *   s_{c,p}[n] = sum_f a_f G_tx G_rx exp(-j 2 pi f0 tau_f)
 *                      rect((t_n - tau_f)/T) exp(j pi K (t_n - tau_f)^2),   t_n = t0[p] + n/fs
 *
 * evaluated term by term in the order O1..O10 of SURVEY.md §8(c), every transcendental
 * through libm in double (long double for frac(f0 tau)), one complex exponential per
 * facet-sample, no recurrences, no tables, no blocking.  The only concession to run time
 * is an OpenMP split of the facet loop with per-thread accumulators (a sum is a sum).
 *
 * Readings of the paper taken here are the G-numbered ones of SURVEY.md §8(c), listed in
 * DESIGN.md §"Readings":  G1 t_n origin, G2 half-open rect and up-chirp, G3 carrier sign,
 * G4 no 1/(r_t r_r), G5 signed field pattern sinc*sinc, G6 cull on |G_t G_r,ref| from the
 * un-offset phase centre, G8 offsets along the Rx unit velocity, G9 stop-and-go,
 * G10 current by advection, G11 linear waves (CWM by flag), G12 tilt factor clamped at 0,
 * G15 A = d^2, G24 displaced point feeds the antenna direction, G27 the generator of the AR(1) speckle innovations
 * (NEXT-1, off unless speckle_tau_s > 0), G28 blending of slopes and velocities on the heterogeneous surface (NEXT-2, off
 * unless wave_nodes_x > 0), G29 bilinear complex antenna patterns on u-v grids (NEXT-3, off unless pattern[k] is given).
 *
 * Pins: tests/test_oracle_pins.py (closed forms with mpmath, invariants, brute force by an
 * independent numpy script).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C0 299792458.0

typedef struct {
    /* instrument */
    double f0_hz, chirp_rate, chirp_len_s, fs_hz;
    int32_t n_samples, n_channels;
    double tx_aperture[2], rx_aperture[2];      /* {azimuth length, elevation height} */
    const double *channel_offset_m;             /* [C] */
    double cull_two_way_db;                     /* <= -300 disables */
    /* geometry */
    int32_t n_pulses;
    const double *t_pulse_s;                    /* [P] */
    const double *tx_pos, *tx_vel, *rx_pos, *rx_vel;   /* [P][3] */
    const double *tx_frame, *rx_frame;          /* [P][3][3] rows: boresight, azimuth, elevation */
    const double *t0_s;                         /* [P] */
    /* scene */
    int32_t nx, ny;
    double spacing_m, centre_m[3];
    int32_t n_waves;
    const double *kx, *ky, *amp, *omega, *phase;/* [Nw] */
    int32_t choppy;
    const float *sigma0_lin;  double sigma0_uniform;   /* [ny][nx] or NULL */
    int32_t tilt_modulation;  double look_dir[2];
    const float *current_mps; double current_uniform[2]; /* [ny][nx][2] or NULL */
    const float *xi;                            /* [ny][nx][2], required */
    /* NEXT-1: time-dependent intra-facet speckle, eq. (7), (10) */
    double speckle_tau_s;                       /* tau_s; <= 0: speckle constant over the dwell (xi)  */
    double speckle_doppler_hz;                  /* f_s of eq. (7)                                      */
    uint64_t seed;                              /* key of the innovation generator (reading G27)       */
    /* NEXT-2: heterogeneous surface, eq. (1), (2).  wave_nodes_x > 0: the wave tables
     * above are ignored; node (a, b) of a lattice of step L whose node (0, 0) sits at the rest position of facet (0, 0)
     * carries its own table of n_waves components -- the homogeneous tile T2L centred on that node. */
    int32_t wave_nodes_x, wave_nodes_y;
    double wave_node_spacing_m;                 /* L */
    const double *node_kx, *node_ky, *node_amp, *node_omega, *node_phase;   /* [nodes_y][nodes_x][n_waves] */
    /* NEXT-3: antenna patterns as complex u-v grids.  pattern[k] non-NULL (k = 0 Tx,
     * 1 Rx) replaces that antenna's analytic sinc pattern: complex field gain on a regular grid of nu x nv nodes
     * over the direction cosines u = r^ . azimuth axis in [u0, u1], v = r^ . elevation axis in [v0, v1]. */
    const float *pattern[2];                    /* [nv][nu][2] (re, im) */
    int32_t pattern_nu[2], pattern_nv[2];
    double pattern_u[2][2], pattern_v[2][2];    /* {first node, last node} */
} oracle_desc;

/* per-facet intermediates of one pulse (O2..O8), exposed for unit parity */
typedef struct {
    double *pos;      /* [F][3]  displaced facet position x_f                */
    double *slope;    /* [F][2]  grad z                                      */
    double *vel;      /* [F][3]  facet velocity (orbital + current)          */
    double *tau;      /* [C][F]  bistatic delay                              */
    double *g_tx;     /* [F]                                                 */
    double *g_rx;     /* [C][F]                                              */
    double *amp;      /* [C][F][2] complex A~ = a G_t G_r exp(-j2pi f0 tau)  */
    int32_t *keep;    /* [F]     1 = survives the cull                       */
} oracle_facets;

static double sinc_pi(double x)
{   /* sin(pi x)/(pi x), sinc(0) = 1  (O6) */
    if (x == 0.0) return 1.0;
    double a = M_PI * x;
    return sin(a) / a;
}

static double dot3(const double *a, const double *b) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }

/* O6: G = sinc(La (u.a)/lambda) sinc(Le (u.e)/lambda), frame rows {b, a, e} */
static double gain(const double *u, const double *frame, const double *aperture, double lambda)
{
    double ua = dot3(u, frame + 3), ue = dot3(u, frame + 6);
    return sinc_pi(aperture[0] * ua / lambda) * sinc_pi(aperture[1] * ue / lambda);
}

/*
 * O6 with tabulated patterns ("antenna patterns are converted into u-v grids at the appropriate
 * resolution"; the gains are complex).  Reading G29: the value between nodes is the bilinear
 * interpolant of the four surrounding nodes, real and imaginary parts separately; a direction outside the grid has
 * zero gain.  Antenna k = 0 is Tx, 1 is Rx; with no table the analytic aperture pattern of `gain` (imaginary part 0).
 */
static void gain_complex(const oracle_desc *d, int k, const double *u, const double *frame, const double *aperture,
                         double lambda, double *re, double *im)
{
    if (!d->pattern[k]) { *re = gain(u, frame, aperture, lambda); *im = 0.0; return; }
    const int nu = d->pattern_nu[k], nv = d->pattern_nv[k];
    const double ua = dot3(u, frame + 3), ue = dot3(u, frame + 6);
    const double gu = (ua - d->pattern_u[k][0]) / (d->pattern_u[k][1] - d->pattern_u[k][0]) * (nu - 1);   /* grid coordinates */
    const double gv = (ue - d->pattern_v[k][0]) / (d->pattern_v[k][1] - d->pattern_v[k][0]) * (nv - 1);
    *re = 0.0; *im = 0.0;
    if (!(gu >= 0.0 && gu <= nu - 1 && gv >= 0.0 && gv <= nv - 1)) return;
    int iu = (int)floor(gu), iv = (int)floor(gv);
    if (iu > nu - 2) iu = nu - 2;
    if (iv > nv - 2) iv = nv - 2;
    const double fu = gu - iu, fv = gv - iv;
    for (int b = 0; b < 2; ++b)
        for (int a = 0; a < 2; ++a) {
            const double wgt = (a ? fu : 1.0 - fu) * (b ? fv : 1.0 - fv);
            const float *t = d->pattern[k] + 2 * ((size_t)(iv + b) * nu + (iu + a));
            *re += wgt * (double)t[0];
            *im += wgt * (double)t[1];
        }
}

typedef struct {
    double pos[3], slope[2], vel[3];
    double tau[8], g_tx, g_rx[8], amp_re[8], amp_im[8];    /* g_tx, g_rx: real parts of the gains */
    int keep;
} facet_eval;

/*
 * Time-dependent intra-facet speckle.  Eq. (7): s(t) = [R(t) + i I(t)] exp(2 i pi f_s t);
 * eq. (10), the order-1 autoregressive model the paper adopts:
 *     R(t + dt) = beta R(t) + (1 - beta^2)^(1/2) R',   beta = exp(-dt / tau_s),   R' ~ N(0, variance 1/2)
 * (the same for I; "sigma = 1/2" of eq. (10) read as the variance, reading G13), started from R(0) + i I(0) = xi_f
 * at pulse 0 and stepped pulse by pulse with dt = t_pulse[q] - t_pulse[q-1].
 * Reading G27 (the paper names no generator): the innovation R' + i I' of facet f at pulse q is drawn from the
 * counter-based generator Philox4x32-10 (Salmon et al., SC'11) with key = the two halves of `seed` and counter
 * (f mod 2^32, f div 2^32, q, 1): with the first two output words w0, w1,
 *     u1 = ((w0 >> 8) + 1) / 2^24 in (0, 1],  u2 = (w1 >> 8) / 2^24 in [0, 1),
 *     R' + i I' = sqrt(-ln u1) (cos 2 pi u2 + i sin 2 pi u2)        (Box-Muller; each part has variance 1/2).
 */
static void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4])
{
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3], k0 = key_in[0], k1 = key_in[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void speckle_innovation(uint64_t seed, uint64_t facet, uint32_t pulse, double *re, double *im)
{
    const uint32_t ctr[4] = { (uint32_t)facet, (uint32_t)(facet >> 32), pulse, 1u };
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    philox4x32_10(ctr, key, w);
    const double u1 = ((double)(w[0] >> 8) + 1.0) / 16777216.0, u2 = (double)(w[1] >> 8) / 16777216.0;
    const double rad = sqrt(-log(u1));
    *re = rad * cos(2.0 * M_PI * u2);
    *im = rad * sin(2.0 * M_PI * u2);
}

/* s_f(t_p) of eq. (7): the AR(1) state after p steps times the intra-facet Doppler factor. */
static void speckle_at(const oracle_desc *d, size_t f, int p, double *re, double *im)
{
    double R = d->xi[2 * f], I = d->xi[2 * f + 1];
    if (d->speckle_tau_s > 0.0) {
        for (int q = 1; q <= p; ++q) {
            const double beta = exp(-(d->t_pulse_s[q] - d->t_pulse_s[q - 1]) / d->speckle_tau_s);
            const double g = sqrt(1.0 - beta * beta);
            double nr, ni;
            speckle_innovation(d->seed, (uint64_t)f, (uint32_t)q, &nr, &ni);
            R = beta * R + g * nr;
            I = beta * I + g * ni;
        }
        const double ph = 2.0 * M_PI * d->speckle_doppler_hz * d->t_pulse_s[p];
        const double c = cos(ph), sn = sin(ph);
        *re = R * c - I * sn;
        *im = R * sn + I * c;
        return;
    }
    *re = R; *im = I;
}

/* O1..O8 for facet (i,j) at pulse p.  Channels limited to 8. */
static void eval_facet(const oracle_desc *d, int p, int i, int j, facet_eval *o)
{
    const double t = d->t_pulse_s[p];
    const double lambda = ORACLE_C0 / d->f0_hz;
    /* O1 rest point */
    double xb = d->centre_m[0] + (i - (d->nx - 1) / 2.0) * d->spacing_m;
    double yb = d->centre_m[1] + (j - (d->ny - 1) / 2.0) * d->spacing_m;
    /* O2 wave sums (linear surface, CWM horizontal displacement by flag).
     * Heterogeneous surface: the displacement at a rest point of the heterogeneous tile TL is the
     * weighted sum of the displacements of the four homogeneous tiles T2L_i centred on TL's corners, eq. (1),
     *     D_TL(x, t) = sum_{i=1..4} W^i(x) D^i_T2L(x, t),
     * with the constant weights of eq. (2),  W^i = (1 - w_x - w_y + w_x w_y)^(1/2),  w_x = |x^i - x|/L, w_y = |y^i - y|/L
     * (their squares add to one).  Reading G28: the same weights blend the facet slope and velocity (the gradient of
     * W itself is not part of the facet orientation). */
    double z = 0, sx = 0, sy = 0, dx = 0, dy = 0, vx = 0, vy = 0, vz = 0;
    const int hetero = d->wave_nodes_x > 0;
    int na = 0, nb = 0;
    double fx = 0, fy = 0;
    if (hetero) {
        const double L = d->wave_node_spacing_m;
        const double ux = i * d->spacing_m / L, uy = j * d->spacing_m / L;     /* lattice coordinates of the rest point */
        na = (int)floor(ux); nb = (int)floor(uy);
        if (na > d->wave_nodes_x - 2) na = d->wave_nodes_x - 2;
        if (nb > d->wave_nodes_y - 2) nb = d->wave_nodes_y - 2;
        fx = ux - na; fy = uy - nb;
    }
    for (int corner = 0; corner < (hetero ? 4 : 1); ++corner) {
        const double *kxs = d->kx, *kys = d->ky, *amps = d->amp, *oms = d->omega, *phs = d->phase;
        double W = 1.0;
        if (hetero) {
            const int ca = corner & 1, cb = corner >> 1;
            const double wx = ca ? 1.0 - fx : fx, wy = cb ? 1.0 - fy : fy;      /* |x^i - x|/L, |y^i - y|/L */
            const double W2 = 1.0 - wx - wy + wx * wy;                            /* eq. (2); = (1 - wx)(1 - wy) >= 0 */
            W = W2 > 0.0 ? sqrt(W2) : 0.0;                                        /* rounding can leave -1e-17 at a far edge */
            const size_t node = ((size_t)(nb + cb) * d->wave_nodes_x + (na + ca)) * d->n_waves;
            kxs = d->node_kx + node; kys = d->node_ky + node; amps = d->node_amp + node;
            oms = d->node_omega + node; phs = d->node_phase + node;
        }
        for (int w = 0; w < d->n_waves; ++w) {
            double k = hypot(kxs[w], kys[w]);
            double psi = kxs[w] * xb + kys[w] * yb - oms[w] * t + phs[w];
            double c = cos(psi), s = sin(psi), a = W * amps[w];
            z  += a * c;
            sx -= a * kxs[w] * s;
            sy -= a * kys[w] * s;
            vz += a * oms[w] * s;
            if (d->choppy && k > 0) {
                dx -= a * kxs[w] / k * s;
                dy -= a * kys[w] / k * s;
                vx += a * oms[w] * kxs[w] / k * c;
                vy += a * oms[w] * kys[w] / k * c;
            }
        }
    }
    double cx = d->current_uniform[0], cy = d->current_uniform[1];
    if (d->current_mps) {
        cx = d->current_mps[((size_t)j * d->nx + i) * 2 + 0];
        cy = d->current_mps[((size_t)j * d->nx + i) * 2 + 1];
    }
    /* O3 displaced position; current by advection (G10; first order = eq. (4)) */
    o->pos[0] = xb + dx + cx * t;
    o->pos[1] = yb + dy + cy * t;
    o->pos[2] = d->centre_m[2] + z;
    o->slope[0] = sx; o->slope[1] = sy;
    o->vel[0] = vx + cx; o->vel[1] = vy + cy; o->vel[2] = vz;
    /* O4 transmit leg */
    const double *ptx = d->tx_pos + 3 * p, *prx = d->rx_pos + 3 * p, *vrx = d->rx_vel + 3 * p;
    double dt[3] = { o->pos[0] - ptx[0], o->pos[1] - ptx[1], o->pos[2] - ptx[2] };
    double rt = sqrt(dot3(dt, dt));
    double ut[3] = { dt[0] / rt, dt[1] / rt, dt[2] / rt };
    double gt_re, gt_im;
    gain_complex(d, 0, ut, d->tx_frame + 9 * p, d->tx_aperture, lambda, &gt_re, &gt_im);
    o->g_tx = gt_re;
    /* O7 cull on the un-offset receive phase centre (G6) */
    double dr0[3] = { o->pos[0] - prx[0], o->pos[1] - prx[1], o->pos[2] - prx[2] };
    double rr0 = sqrt(dot3(dr0, dr0));
    double ur0[3] = { dr0[0] / rr0, dr0[1] / rr0, dr0[2] / rr0 };
    double gref_re, gref_im;
    gain_complex(d, 1, ur0, d->rx_frame + 9 * p, d->rx_aperture, lambda, &gref_re, &gref_im);
    o->keep = 1;
    if (d->cull_two_way_db > -300.0) {
        double thr = pow(10.0, d->cull_two_way_db / 20.0);
        if (hypot(gt_re, gt_im) * hypot(gref_re, gref_im) < thr) o->keep = 0;       /* |G_t G_r,ref| */
    }
    /* O8 amplitude a = sqrt(sigma d^2) xi   (G15, G12) */
    double sigma = d->sigma0_lin ? (double)d->sigma0_lin[(size_t)j * d->nx + i] : d->sigma0_uniform;
    if (d->tilt_modulation) {
        double f = 1.0 + 2.0 * (sx * d->look_dir[0] + sy * d->look_dir[1]);
        sigma *= (f > 0.0 ? f : 0.0);
    }
    double a0 = sqrt(sigma * d->spacing_m * d->spacing_m);
    double xr, xim;
    speckle_at(d, (size_t)j * d->nx + i, p, &xr, &xim);
    double vn = sqrt(dot3(vrx, vrx));
    for (int c = 0; c < d->n_channels; ++c) {
        /* O4 receive leg: phase centre offset along the Rx unit velocity (G8) */
        double pc[3] = { prx[0] + d->channel_offset_m[c] * vrx[0] / vn,
                         prx[1] + d->channel_offset_m[c] * vrx[1] / vn,
                         prx[2] + d->channel_offset_m[c] * vrx[2] / vn };
        double dr[3] = { o->pos[0] - pc[0], o->pos[1] - pc[1], o->pos[2] - pc[2] };
        double rr = sqrt(dot3(dr, dr));
        double ur[3] = { dr[0] / rr, dr[1] / rr, dr[2] / rr };
        double gr_re, gr_im;
        gain_complex(d, 1, ur, d->rx_frame + 9 * p, d->rx_aperture, lambda, &gr_re, &gr_im);
        /* O5 */
        double tau = (rt + rr) / ORACLE_C0;
        /* carrier phase -2 pi frac(f0 tau), long double for the 2.8e7-cycle product (G3) */
        long double cyc = (long double)d->f0_hz * (long double)tau;
        double fr = (double)(cyc - floorl(cyc));
        double ph = -2.0 * M_PI * fr;
        /* a G_t G_r: complex product of the two gains, then of the speckle */
        double g_re = a0 * (gt_re * gr_re - gt_im * gr_im), g_im = a0 * (gt_re * gr_im + gt_im * gr_re);
        double ar = g_re * xr - g_im * xim, ai = g_re * xim + g_im * xr;
        o->tau[c] = tau;
        o->g_rx[c] = gr_re;
        o->amp_re[c] = ar * cos(ph) - ai * sin(ph);
        o->amp_im[c] = ar * sin(ph) + ai * cos(ph);
    }
}

/* O9: add one facet-echo into acc[Ns][2] (interleaved re, im). */
static void add_echo(const oracle_desc *d, int p, double tau, double are, double aim, double *acc)
{
    const double T = d->chirp_len_s, K = d->chirp_rate, fs = d->fs_hz, t0 = d->t0_s[p];
    /* candidate samples: everything within one sample of the replica support */
    double centre = (tau - t0) * fs;
    long n_lo = (long)floor(centre - 0.5 * T * fs) - 2;
    long n_hi = (long)ceil(centre + 0.5 * T * fs) + 2;
    if (n_lo < 0) n_lo = 0;
    if (n_hi > d->n_samples - 1) n_hi = d->n_samples - 1;
    for (long n = n_lo; n <= n_hi; ++n) {
        double u = (t0 + (double)n / fs) - tau;
        if (u >= -0.5 * T && u < 0.5 * T) {           /* rect, half-open (G2) */
            double ph = M_PI * K * u * u;
            double c = cos(ph), s = sin(ph);
            acc[2 * n]     += are * c - aim * s;
            acc[2 * n + 1] += are * s + aim * c;
        }
    }
}

/*
 * heeps_oracle_generate: out[C][n_sel][Ns][2] (double re,im) for the listed pulses.
 * Returns 0, or -1 on bad arguments.
 */
int heeps_oracle_generate(const oracle_desc *d, const int32_t *pulses, int32_t n_sel, double *out,
                          int32_t n_threads)
{
    if (!d || !pulses || !out || d->n_channels < 1 || d->n_channels > 8 || !d->xi) return -1;
    const int C = d->n_channels, Ns = d->n_samples;
    const size_t vec = (size_t)Ns * 2;
    memset(out, 0, sizeof(double) * vec * C * n_sel);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    for (int s = 0; s < n_sel; ++s) {
        const int p = pulses[s];
        if (p < 0 || p >= d->n_pulses) return -1;
#pragma omp parallel
        {
            double *acc = (double *)calloc(vec * C, sizeof(double));
#pragma omp for schedule(static)
            for (int j = 0; j < d->ny; ++j) {
                for (int i = 0; i < d->nx; ++i) {
                    facet_eval fe;
                    eval_facet(d, p, i, j, &fe);
                    if (!fe.keep) continue;                       /* O7 */
                    for (int c = 0; c < C; ++c)
                        add_echo(d, p, fe.tau[c], fe.amp_re[c], fe.amp_im[c], acc + vec * c);
                }
            }
#pragma omp critical
            {
                for (int c = 0; c < C; ++c) {
                    double *o = out + ((size_t)c * n_sel + s) * vec;
                    for (size_t k = 0; k < vec; ++k) o[k] += acc[vec * c + k];
                }
            }
            free(acc);
        }
    }
    return 0;
}

/*
 * heeps_oracle_samples: the same defined sum, but only for the listed output samples n_list[0..count)
 * of one pulse: out[C][count][2].  Lets the tests check full-size configurations sample by sample
 * (every facet is still evaluated; only the O9 loop is restricted to the listed n).
 */
int heeps_oracle_samples(const oracle_desc *d, int32_t p, const int32_t *n_list, int32_t count, double *out,
                         int32_t n_threads)
{
    if (!d || !n_list || !out || p < 0 || p >= d->n_pulses || d->n_channels > 8 || !d->xi || count < 1) return -1;
    const int C = d->n_channels;
    const double T = d->chirp_len_s, K = d->chirp_rate, fs = d->fs_hz, t0 = d->t0_s[p];
    memset(out, 0, sizeof(double) * 2 * C * count);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel
    {
        double *acc = (double *)calloc((size_t)2 * C * count, sizeof(double));
#pragma omp for schedule(static)
        for (int j = 0; j < d->ny; ++j)
            for (int i = 0; i < d->nx; ++i) {
                facet_eval fe;
                eval_facet(d, p, i, j, &fe);
                if (!fe.keep) continue;
                for (int c = 0; c < C; ++c)
                    for (int q = 0; q < count; ++q) {
                        double u = (t0 + (double)n_list[q] / fs) - fe.tau[c];
                        if (u >= -0.5 * T && u < 0.5 * T) {
                            double ph = M_PI * K * u * u;
                            double cs = cos(ph), sn = sin(ph);
                            acc[2 * (c * count + q)]     += fe.amp_re[c] * cs - fe.amp_im[c] * sn;
                            acc[2 * (c * count + q) + 1] += fe.amp_re[c] * sn + fe.amp_im[c] * cs;
                        }
                    }
            }
#pragma omp critical
        for (int k = 0; k < 2 * C * count; ++k) out[k] += acc[k];
        free(acc);
    }
    return 0;
}

/* heeps_oracle_facets: O2..O8 intermediates of one pulse (any pointer may be NULL). */
int heeps_oracle_facets(const oracle_desc *d, int32_t p, oracle_facets *o)
{
    if (!d || !o || p < 0 || p >= d->n_pulses || d->n_channels > 8 || !d->xi) return -1;
    const size_t F = (size_t)d->nx * d->ny;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < d->ny; ++j)
        for (int i = 0; i < d->nx; ++i) {
            facet_eval fe;
            eval_facet(d, p, i, j, &fe);
            size_t f = (size_t)j * d->nx + i;
            if (o->pos)   for (int k = 0; k < 3; ++k) o->pos[3 * f + k] = fe.pos[k];
            if (o->slope) for (int k = 0; k < 2; ++k) o->slope[2 * f + k] = fe.slope[k];
            if (o->vel)   for (int k = 0; k < 3; ++k) o->vel[3 * f + k] = fe.vel[k];
            if (o->g_tx)  o->g_tx[f] = fe.g_tx;
            if (o->keep)  o->keep[f] = fe.keep;
            for (int c = 0; c < d->n_channels; ++c) {
                if (o->tau)  o->tau[c * F + f] = fe.tau[c];
                if (o->g_rx) o->g_rx[c * F + f] = fe.g_rx[c];
                if (o->amp) { o->amp[2 * (c * F + f)] = fe.amp_re[c]; o->amp[2 * (c * F + f) + 1] = fe.amp_im[c]; }
            }
        }
    return 0;
}

/* heeps_oracle_philox: the raw generator (for its known-answer pins). */
void heeps_oracle_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }

/* heeps_oracle_speckle: s_f(t_p) of every facet at pulse p, out[F][2]. */
int heeps_oracle_speckle(const oracle_desc *d, int32_t p, double *out)
{
    if (!d || !out || p < 0 || p >= d->n_pulses || !d->xi) return -1;
    const size_t F = (size_t)d->nx * d->ny;
#pragma omp parallel for schedule(static)
    for (long f = 0; f < (long)F; ++f) speckle_at(d, (size_t)f, p, out + 2 * f, out + 2 * f + 1);
    return 0;
}

int heeps_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
