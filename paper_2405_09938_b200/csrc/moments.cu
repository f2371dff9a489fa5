// K2s -- geometry, gains, amplitude, cull and RANGE-SLICE MOMENTS for the spectral path
// (SURVEY.md §8(a) A2..A5 and the "Moment form" of A6; "the complex amplitudes of
// all facets lying in range slices R_i <= r_t + r_r <= R_{i+1} (eq. 17) are added to obtain one time
// sample ... the obtained profile can be regarded as the impulse response of the surface and
// subsequently convolved by the waveform").
//
// The paper's plain slice sum drops the position of a facet inside its slice; at one slice per sample
// that is 0.4 relative L2 away from the defined sum.  Here the sub-slice position
// eps in [0,1) is kept to any order: with b = ceil(nu) (integer slice = first in-window sample),
// m = n - b, y = 2 eps - 1 and z_m = 2 pi kappa (m - L/2),
//
//   g_m(y) = exp(j 2 pi kappa (m + eps - L/2)^2) = sum_k c_k[m] T_k(y)        (Chebyshev series in y of the slice response;
//            = exp(j 2 pi kappa ((m-L/2)^2 + (m-L/2) + eps^2)) exp(j z_m y), whose last factor is the Jacobi-Anger series
//            sum_k e_k j^k J_k(z_m) T_k(y), |z_m| <= pi B/(2 fs); sim_api.cu computes c_k[m] by quadrature)
//
// so  s[n] = sum_{k<Kt} sum_m c_k[m] M_k[n-m]  with the Chebyshev moments of each slice
//
//   M_k[b] = sum_{f: b_f = b} |A~_f| exp(j 2 pi (-dR_f/lambda + arg A~_f)) T_k(y_f)
//
// (Kt = 1 is eq. (17) with the slice response at its mean; Kt = 8 truncates at J_8(1.31) ~ 1e-6; sim_create refuses the
// form when the tail beyond Kt exceeds 5e-6.)  This kernel produces M; the
// convolution with the Kt waveform kernels c_k is fftconv.cu.
//
// One CTA = one spatial tile (<= 32 x 32 facets) of one pulse.  Facet state (fp64 position, Tx leg, cull)
// is computed once and kept in registers; per channel the facet-echoes are counting-sorted by slice in
// shared memory (integer ATOMS on a histogram -- shared FP32 atomics would be CAS loops), then 8 threads
// per slice sum the slice's Kt complex moments, exchange them with a 3-level shuffle reduce-scatter and
// issue ONE vector RED.ADD.F32x2 per (slice, k) to the global moment rows.
//
// Bound: FP64 pipe (ranges) + FP32; HBM: 8 B z + maps read per facet-pulse, nothing written per facet-echo.
#include "kernels.cuh"
#include "geometry_common.cuh"

namespace heeps {

namespace {

constexpr int kThreads = 256;
constexpr int kKt = kMomentOrder;      // 8
static_assert(kKt == 8, "the reduce-scatter below is written for 8 moments / 8 threads per slice");

template <int FPT, bool kSeries>
__global__ void __launch_bounds__(kThreads)
moments_kernel(DevParams prm, MomentArgs a, int p0, int n_pl)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ PulseConst pc;
    __shared__ int s_base[kMaxChannels];
    __shared__ unsigned long long s_samples;
    __shared__ int s_kept;

    const int span = a.span_cap;
    float4 *payload = reinterpret_cast<float4 *>(smem_raw);                 // [tile_cap] sorted by slice
    int *hist = reinterpret_cast<int *>(smem_raw + (size_t)prm.tile_cap * 16);   // [span + 1]

    const int tile = blockIdx.x, pl = blockIdx.y, p = p0 + pl;
    const int tid = threadIdx.x, lane = tid & 31;
    {
        const double *src = reinterpret_cast<const double *>(a.pulses + p);
        double *dst = reinterpret_cast<double *>(&pc);
        for (int k = tid; k < (int)(sizeof(PulseConst) / sizeof(double)); k += kThreads) dst[k] = src[k];
    }
    if (tid == 0) { s_samples = 0ull; s_kept = 0; }
    __syncthreads();

    const int C = prm.n_channels, ts = prm.tile, L = a.replica;
    const int ti0 = (tile % prm.tiles_x) * ts, tj0 = (tile / prm.tiles_x) * ts;
    if (tid < C) {
        // slice window of this (tile, pulse, channel): centred on the slice of the tile centre (rest, flat)
        const double ic = ti0 + 0.5 * (min(ts, prm.nx - ti0) - 1), jc = tj0 + 0.5 * (min(ts, prm.ny - tj0) - 1);
        const double x = prm.cx + (ic - 0.5 * (prm.nx - 1)) * prm.spacing;
        const double y = prm.cy + (jc - 0.5 * (prm.ny - 1)) * prm.spacing;
        const double ax = x - pc.tx_pos[0], ay = y - pc.tx_pos[1], az = prm.cz - pc.tx_pos[2];
        const double bx = x - pc.rx_pos[tid][0], by = y - pc.rx_pos[tid][1], bz = prm.cz - pc.rx_pos[tid][2];
        const double dR = sqrt(ax * ax + ay * ay + az * az) + sqrt(bx * bx + by * by + bz * bz) - pc.r0;
        double bc = ceil(dR * prm.fs_over_c0 - prm.half_len) - 0.5 * span;
        bc = fmin(fmax(bc, -1.0e9), 1.0e9);
        s_base[tid] = (int)bc;
    }

    // ---- facet state, once for all channels (O1..O3, Tx leg, cull reference, amplitude) ----
    const size_t F = (size_t)prm.nx * prm.ny;
    const SurfaceInterp it = surface_interp(a.surf, a.pulses, p, pl);
    const float area = (float)(prm.spacing * prm.spacing);
    double pos[FPT][3], rt[FPT], dv[FPT];
    LegParts ref[FPT];
    float gt[FPT], amag[FPT];
    float gti[FPT];                                      // Im G_t (tabulated patterns only)
    uint32_t xarg[FPT];
    bool keep[FPT];
    int my_kept = 0;
#pragma unroll
    for (int q = 0; q < FPT; ++q) {
        const int k = q * kThreads + tid;
        const int li = k % ts, lj = k / ts;
        const int i = ti0 + li, j = tj0 + lj;
        keep[q] = false;
        rt[q] = 0.0; gt[q] = 0.f; gti[q] = 0.f; amag[q] = 0.f; xarg[q] = 0u;
        pos[q][0] = pos[q][1] = pos[q][2] = 0.0;
        if (k < ts * ts && i < prm.nx && j < prm.ny) {
            const size_t f = (size_t)j * prm.nx + i;
            const double xb = prm.cx + ((double)i - 0.5 * (prm.nx - 1)) * prm.spacing;
            const double yb = prm.cy + ((double)j - 0.5 * (prm.ny - 1)) * prm.spacing;
            double cux = prm.cur_ux, cuy = prm.cur_uy;
            if (a.current) { const float2 cv = __ldg(a.current + f); cux = cv.x; cuy = cv.y; }
            pos[q][0] = xb + cux * pc.t;
            pos[q][1] = yb + cuy * pc.t;
            pos[q][2] = prm.cz + surface_z(a.surf, it, F, f);
            if (a.surf.dxy) { const double2 dd = surface_dxy(a.surf, it, F, f); pos[q][0] += dd.x; pos[q][1] += dd.y; }
            const LegParts lt = leg_parts(pos[q], pc.tx_pos, pc.tx_a, pc.tx_e);
            ref[q] = leg_parts(pos[q], pc.rx_ref, pc.rx_a, pc.rx_e);
            dv[q] = fma(ref[q].dx, pc.rx_vhat[0], fma(ref[q].dy, pc.rx_vhat[1], ref[q].dz * pc.rx_vhat[2]));
            rt[q] = lt.r; gt[q] = pattern(lt.da, lt.de, lt.inv, prm.ap_tx_a, prm.ap_tx_e);
            const float g_ref = pattern(ref[q].da, ref[q].de, ref[q].inv, prm.ap_rx_a, prm.ap_rx_e);
            keep[q] = !(fabsf(gt[q] * g_ref) < prm.cull_thr);               // O7 (G6)
            if (prm.lut_any) {                                              // tabulated patterns: complex gains
                const float2 gtc = gain_of(prm, 0, gt[q], lt.da * lt.inv, lt.de * lt.inv);
                const float2 grc = gain_of(prm, 1, g_ref, ref[q].da * ref[q].inv, ref[q].de * ref[q].inv);
                gt[q] = gtc.x; gti[q] = gtc.y;
                keep[q] = !(hypotf(gtc.x, gtc.y) * hypotf(grc.x, grc.y) < prm.cull_thr);
            }
            float sig = a.sigma0 ? __ldg(a.sigma0 + f) : (float)prm.sigma0_uniform;
            if (prm.tilt) {
                const float2 sl = surface_slope(a.surf, it, F, f);
                sig *= fmaxf(1.f + 2.f * (sl.x * (float)prm.look_x + sl.y * (float)prm.look_y), 0.f);
            }
            const uint2 xp = __ldg(a.xi_polar + (size_t)pl * a.xi_pulse_stride + f);
            amag[q] = sqrtf(sig * area) * __uint_as_float(xp.x);           // |a_f| (O8)
            xarg[q] = xp.y;
            if (keep[q]) ++my_kept;
        }
    }
    unsigned long long my_samples = 0;

    for (int c = 0; c < C; ++c) {
        for (int k = tid; k <= span; k += kThreads) hist[k] = 0;
        __syncthreads();                                   // also publishes s_base
        const int base = s_base[c];

        // ---- per facet-echo: slice, sub-slice position, complex weight; rank inside the slice ----
        float br[FPT], bi[FPT], yy[FPT];
        int bin[FPT], rank[FPT];
#pragma unroll
        for (int q = 0; q < FPT; ++q) {
            bin[q] = -1; rank[q] = 0; br[q] = bi[q] = yy[q] = 0.f;
            if (!keep[q]) continue;
            double r_c, inv_c, da_c, de_c;
            if (kSeries) {
                channel_leg_series(ref[q], dv[q], pc.ch_off[c], pc.rx_va, pc.rx_ve, r_c, inv_c, da_c, de_c);
            } else {
                const LegParts lc = leg_parts(pos[q], pc.rx_pos[c], pc.rx_a, pc.rx_e);
                r_c = lc.r; inv_c = lc.inv; da_c = lc.da; de_c = lc.de;
            }
            const float g_rx = pattern(da_c, de_c, inv_c, prm.ap_rx_a, prm.ap_rx_e);
            const double dR = (rt[q] + r_c) - pc.r0;
            const double nu = dR * prm.fs_over_c0 - prm.half_len;
            const double bd = ceil(nu);
            if (!(bd > -(double)L && bd < (double)prm.n_samples)) continue;    // window misses [0, Ns)
            const int b = (int)bd;
            const double eps = bd - nu;                                    // [0, 1)
            const float g = gt[q] * g_rx;
            const uint32_t garg = (g < 0.f && !prm.lut_any) ? 0x80000000u : 0u;
            const uint32_t ph = turns_to_u32_fast(-dR * prm.inv_lambda) + xarg[q] + garg;    // (the chirp's kappa eps^2 is part of c_k)
            float sn, cs;
            __sincosf((float)(int32_t)ph * 1.4629180792671596e-9f, &sn, &cs);   // 2 pi / 2^32
            if (prm.lut_any) {                                             // complex gain product times the phasor
                const float2 cg = cmulf(make_float2(gt[q], gti[q]), gain_of(prm, 1, g_rx, da_c * inv_c, de_c * inv_c));
                const float2 w = cmulf(cg, make_float2(cs, sn));
                br[q] = amag[q] * w.x; bi[q] = amag[q] * w.y;
            } else {
                const float mag = fabsf(g) * amag[q];
                br[q] = mag * cs; bi[q] = mag * sn;
            }
            yy[q] = (float)(2.0 * eps - 1.0);
            my_samples += (unsigned)(min(b + L, prm.n_samples) - max(b, 0));
            const int rel = b - base;
            if (rel >= 0 && rel < span) {
                bin[q] = rel;
                rank[q] = atomicAdd(&hist[rel + 1], 1);
            } else {                                                       // outside the tile window: rare
                float2 *row = a.mom + ((size_t)(c * n_pl + pl) * kKt) * a.nb_pad + (b + L - 1);
                float t0 = 1.f, t1 = yy[q];
                atomicAdd(row, make_float2(br[q], bi[q]));
                atomicAdd(row + a.nb_pad, make_float2(br[q] * t1, bi[q] * t1));
                for (int k = 2; k < kKt; ++k) {
                    const float t2 = 2.f * yy[q] * t1 - t0;
                    atomicAdd(row + (size_t)k * a.nb_pad, make_float2(br[q] * t2, bi[q] * t2));
                    t0 = t1; t1 = t2;
                }
            }
        }
        __syncthreads();
        if (tid < 32) {                                     // inclusive scan of hist[1..span] by one warp
            int carry = 0;
            for (int k0 = 1; k0 <= span; k0 += 32) {
                const int k = k0 + lane;
                int v = (k <= span) ? hist[k] : 0;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int t = __shfl_up_sync(0xffffffffu, v, o);
                    if (lane >= o) v += t;
                }
                if (k <= span) hist[k] = v + carry;
                carry += __shfl_sync(0xffffffffu, v, 31);
            }
        }
        __syncthreads();                                    // hist[s] = first sorted position of slice s
#pragma unroll
        for (int q = 0; q < FPT; ++q)
            if (bin[q] >= 0) payload[hist[bin[q]] + rank[q]] = make_float4(br[q], bi[q], yy[q], 0.f);
        __syncthreads();

        // ---- 8 threads per slice: Chebyshev moments of the slice, reduce-scatter, one RED per (slice, k) ----
        const int sub = tid & 7;
        for (int s0 = 0; s0 < span; s0 += kThreads / 8) {
            const int s = s0 + (tid >> 3);
            int first = 0, cnt = 0;
            if (s < span) { first = hist[s]; cnt = hist[s + 1] - first; }
            if (__ballot_sync(0xffffffffu, cnt > 0) == 0u) continue;       // warp-uniform
            float2 m[kKt];
#pragma unroll
            for (int k = 0; k < kKt; ++k) m[k] = make_float2(0.f, 0.f);
            for (int i = sub; i < cnt; i += 8) {
                const float4 v = payload[first + i];
                const float y2 = v.z + v.z;
                float t0 = 1.f, t1 = v.z;
                m[0].x += v.x; m[0].y += v.y;
                m[1].x = fmaf(v.x, t1, m[1].x); m[1].y = fmaf(v.y, t1, m[1].y);
#pragma unroll
                for (int k = 2; k < kKt; ++k) {
                    const float t2 = fmaf(y2, t1, -t0);
                    m[k].x = fmaf(v.x, t2, m[k].x); m[k].y = fmaf(v.y, t2, m[k].y);
                    t0 = t1; t1 = t2;
                }
            }
            // reduce-scatter over the 8 threads of the slice: thread `sub` ends with moment k = sub
            float2 h4[4], h2[2], h1;
            {
                const bool hi = sub & 4;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const float2 send = hi ? m[k] : m[k + 4], kp = hi ? m[k + 4] : m[k];
                    h4[k].x = kp.x + __shfl_xor_sync(0xffffffffu, send.x, 4);
                    h4[k].y = kp.y + __shfl_xor_sync(0xffffffffu, send.y, 4);
                }
            }
            {
                const bool hi = sub & 2;
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const float2 send = hi ? h4[k] : h4[k + 2], kp = hi ? h4[k + 2] : h4[k];
                    h2[k].x = kp.x + __shfl_xor_sync(0xffffffffu, send.x, 2);
                    h2[k].y = kp.y + __shfl_xor_sync(0xffffffffu, send.y, 2);
                }
            }
            {
                const bool hi = sub & 1;
                const float2 send = hi ? h2[0] : h2[1], kp = hi ? h2[1] : h2[0];
                h1.x = kp.x + __shfl_xor_sync(0xffffffffu, send.x, 1);
                h1.y = kp.y + __shfl_xor_sync(0xffffffffu, send.y, 1);
            }
            if (cnt > 0) {
                float2 *row = a.mom + ((size_t)(c * n_pl + pl) * kKt + sub) * a.nb_pad;
                atomicAdd(row + (base + s + L - 1), h1);
            }
        }
        __syncthreads();                                    // hist / payload are reused by the next channel
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
}

}  // namespace

size_t moments_smem_bytes(const DevParams &prm, int span_cap)
{
    return (size_t)prm.tile_cap * 16 + (size_t)(span_cap + 1) * 4;
}

cudaError_t launch_moments(const DevParams &prm, const MomentArgs &a, int p0, int n_pl, cudaStream_t s)
{
    dim3 grid(prm.n_tiles, n_pl);
    const size_t smem = moments_smem_bytes(prm, a.span_cap);
    const bool series = prm.series_channels != 0;
    if (prm.tile_cap <= kThreads) {
        if (series) moments_kernel<1, true><<<grid, kThreads, smem, s>>>(prm, a, p0, n_pl);
        else        moments_kernel<1, false><<<grid, kThreads, smem, s>>>(prm, a, p0, n_pl);
    } else if (prm.tile_cap <= 4 * kThreads) {
        if (series) moments_kernel<4, true><<<grid, kThreads, smem, s>>>(prm, a, p0, n_pl);
        else        moments_kernel<4, false><<<grid, kThreads, smem, s>>>(prm, a, p0, n_pl);
    } else {
        return cudaErrorInvalidValue;      // the spectral path tiles at <= 32 x 32 facets
    }
    return cudaGetLastError();
}

}  // namespace heeps
