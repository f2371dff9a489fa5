// K2 -- bistatic geometry, antenna gains, scattering amplitude, cull, tile bucketing
// (SURVEY.md §8(a) A2..A5; PAPER.md:91-98 ranges and geometric phase, :202 antenna patterns
// evaluated "at each facet and for each pulse", :223 contributing subset per pulse).
//
// One block = one spatial tile of one pulse.  Ranges, the echo centre, the integer window
// [b, b+cnt) and both phase coefficients are computed in fp64 (1 mrad = 8.8 um of path); the
// result handed to K3 is a 32-byte record whose phase is 32-bit fixed point in turns, so K3
// never touches a large floating-point phase.  Surviving facets of a tile are compacted in
// facet order with a block scan (deterministic), one record list per channel; the per-tile
// sample span (min first sample, max end sample) replaces a global delay sort: a spatial tile
// is already narrow in delay (SURVEY.md §8(a) A5 "tile-local bins").
//
// Bound: FP64 pipe (~60 DFMA per facet-antenna) + 32 B written per surviving facet-echo.
#include "kernels.cuh"
#include "geometry_common.cuh"

namespace heeps {

namespace {

constexpr int kThreads = 256;

template <bool kDebug>
__global__ void __launch_bounds__(kThreads)
geometry_kernel(DevParams prm, GeometryArgs a, int p0, int n_pl)
{
    __shared__ PulseConst pc;
    __shared__ int s_warp_cnt[kThreads / 32];
    __shared__ int s_base;
    __shared__ int s_bmin[kMaxChannels], s_bmax[kMaxChannels];
    __shared__ unsigned long long s_samples;
    __shared__ uint32_t s_shift[kMaxChannels];

    const int tile = blockIdx.x, pl = blockIdx.y, p = p0 + pl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    {   // broadcast the pulse constants
        const double *src = reinterpret_cast<const double *>(a.pulses + p);
        double *dst = reinterpret_cast<double *>(&pc);
        for (int k = tid; k < (int)(sizeof(PulseConst) / sizeof(double)); k += kThreads) dst[k] = src[k];
    }
    if (tid == 0) { s_base = 0; s_samples = 0ull; }
    if (tid < kMaxChannels) { s_bmin[tid] = INT_MAX; s_bmax[tid] = INT_MIN; }
    __syncthreads();

    const int C = prm.n_channels, ts = prm.tile;
    const int ti0 = (tile % prm.tiles_x) * ts, tj0 = (tile / prm.tiles_x) * ts;
    if (tid < C) {
        // frequency shift of this (tile, pulse, channel): a quarter cycle per sample minus the dechirped
        // tone frequency of the tile centre (rest position, flat surface)
        const double ic = ti0 + 0.5 * (min(ts, prm.nx - ti0) - 1), jc = tj0 + 0.5 * (min(ts, prm.ny - tj0) - 1);
        const double x = prm.cx + (ic - 0.5 * (prm.nx - 1)) * prm.spacing;
        const double y = prm.cy + (jc - 0.5 * (prm.ny - 1)) * prm.spacing;
        const double ax = x - pc.tx_pos[0], ay = y - pc.tx_pos[1], az = prm.cz - pc.tx_pos[2];
        const double bx = x - pc.rx_pos[tid][0], by = y - pc.rx_pos[tid][1], bz = prm.cz - pc.rx_pos[tid][2];
        const double dR = sqrt(ax * ax + ay * ay + az * az) + sqrt(bx * bx + by * by + bz * bz) - pc.r0;
        const double cpc = dR * prm.fs_over_c0 - (double)prm.n_mid;
        s_shift[tid] = turns_to_u32(0.25 + 2.0 * prm.kappa * cpc);
    }
    __syncthreads();
    const size_t F = (size_t)prm.nx * prm.ny;
    const SurfaceInterp it = surface_interp(a.surf, a.pulses, p, pl);
    const float area = (float)(prm.spacing * prm.spacing);
    unsigned long long my_samples = 0;
    int my_bmin[kMaxChannels], my_bmax[kMaxChannels];
#pragma unroll
    for (int c = 0; c < kMaxChannels; ++c) { my_bmin[c] = INT_MAX; my_bmax[c] = INT_MIN; }

    for (int k0 = 0; k0 < ts * ts; k0 += kThreads) {
        const int k = k0 + tid;
        const int li = k % ts, lj = k / ts;
        const int i = ti0 + li, j = tj0 + lj;
        const bool valid = (k < ts * ts) && i < prm.nx && j < prm.ny;
        bool keep = false;
        double pos[3] = {0, 0, 0};
        float gt = 0.f, a0 = 0.f;
        float2 gtc = make_float2(0.f, 0.f);                  // complex Tx gain (tabulated patterns only)
        double rt = 0;
        float2 xi = make_float2(0.f, 0.f);
        float xi_mag = 0.f;
        uint32_t xi_arg = 0u;
        size_t f = 0;
        if (valid) {
            f = (size_t)j * prm.nx + i;
            // O1 rest point, O3 displaced position (current by advection, G10)
            double xb = prm.cx + ((double)i - 0.5 * (prm.nx - 1)) * prm.spacing;
            double yb = prm.cy + ((double)j - 0.5 * (prm.ny - 1)) * prm.spacing;
            double cux = prm.cur_ux, cuy = prm.cur_uy;
            if (a.current) { float2 cv = __ldg(a.current + f); cux = cv.x; cuy = cv.y; }
            pos[0] = xb + cux * pc.t;
            pos[1] = yb + cuy * pc.t;
            pos[2] = prm.cz + surface_z(a.surf, it, F, f);
            if (a.surf.dxy) { double2 dd = surface_dxy(a.surf, it, F, f); pos[0] += dd.x; pos[1] += dd.y; }
            // O4/O6 transmit leg and the cull reference (G6)
            Leg lt = leg(pos, pc.tx_pos, pc.tx_a, pc.tx_e, prm.ap_tx_a, prm.ap_tx_e);
            Leg lr = leg(pos, pc.rx_ref, pc.rx_a, pc.rx_e, prm.ap_rx_a, prm.ap_rx_e);
            rt = lt.r; gt = lt.g;
            keep = !(fabsf(gt * lr.g) < prm.cull_thr);
            if (prm.lut_any) {                               // tabulated patterns: complex gains, cull on |G_t| |G_r,ref|
                gtc = gain_of(prm, 0, lt.g, lt.ua, lt.ue);
                const float2 grc = gain_of(prm, 1, lr.g, lr.ua, lr.ue);
                gt = gtc.x;
                keep = !(hypotf(gtc.x, gtc.y) * hypotf(grc.x, grc.y) < prm.cull_thr);
            }
            // O8 amplitude
            float sig = a.sigma0 ? __ldg(a.sigma0 + f) : (float)prm.sigma0_uniform;
            if (prm.tilt) {
                float2 sl = surface_slope(a.surf, it, F, f);
                float fac = 1.f + 2.f * (sl.x * (float)prm.look_x + sl.y * (float)prm.look_y);
                sig *= fmaxf(fac, 0.f);
            }
            a0 = sqrtf(sig * area);
            { uint2 xp = __ldg(a.xi_polar + (size_t)pl * a.xi_pulse_stride + f); xi_mag = __uint_as_float(xp.x); xi_arg = xp.y; }
            if (!a.xi_pulse_stride) xi = __ldg(a.xi + f);
            else if (a.dbg_amp) {                            // time-dependent speckle: the complex value for the report
                double sn, cs;
                sincospi(2.0 * (double)xi_arg * 2.3283064365386963e-10, &sn, &cs);
                xi = make_float2((float)(xi_mag * cs), (float)(xi_mag * sn));
            }
            if (kDebug) {
                if (a.dbg_pos) { a.dbg_pos[3 * f] = pos[0]; a.dbg_pos[3 * f + 1] = pos[1]; a.dbg_pos[3 * f + 2] = pos[2]; }
                if (a.dbg_gtx) a.dbg_gtx[f] = gt;
                if (a.dbg_keep) a.dbg_keep[f] = keep ? 1 : 0;
            }
        }
        // deterministic block compaction of the survivors (facet order)
        const unsigned bal = __ballot_sync(0xffffffffu, keep);
        if (lane == 0) s_warp_cnt[warp] = __popc(bal);
        __syncthreads();
        int idx = s_base + __popc(bal & ((1u << lane) - 1u));
        int total = 0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) {
            int cnt = s_warp_cnt[w];
            if (w < warp) idx += cnt;
            total += cnt;
        }
        __syncthreads();
        if (tid == 0) s_base += total;

        if (valid && (keep || kDebug)) {
            for (int c = 0; c < C; ++c) {
                Leg lr = leg(pos, pc.rx_pos[c], pc.rx_a, pc.rx_e, prm.ap_rx_a, prm.ap_rx_e);
                const double dR = (rt + lr.r) - pc.r0;            // path beyond sample 0
                const double cs = dR * prm.fs_over_c0;            // echo centre [samples]
                const double cp = cs - (double)prm.n_mid;
                const double nu = cs - prm.half_len;
                const int b = (int)ceil(nu);
                const int e = (int)ceil(nu + prm.len);
                float g = a0 * gt * lr.g;
                float2 cg = make_float2(g, 0.f);                   // a G_t G_r,c
                uint32_t garg = (gt * lr.g < 0.f) ? 0x80000000u : 0u;
                float grx_re = lr.g;
                if (prm.lut_any) {
                    const float2 grc = gain_of(prm, 1, lr.g, lr.ua, lr.ue);
                    const float2 pr = cmulf(gtc, grc);
                    cg = make_float2(a0 * pr.x, a0 * pr.y);
                    g = hypotf(cg.x, cg.y);
                    garg = arg_u32(cg);
                    grx_re = grc.x;
                }
                if (keep) {
                    Rec r;
                    // arg(A~) = arg(xi) (+ half a turn when G_t G_r < 0): exact adds on the phase word
                    r.phi = turns_to_u32(fma(prm.kappa * cp, cp, -dR * prm.inv_lambda)) + kPhiBias + xi_arg + garg;
                    r.beta = turns_to_u32(-2.0 * prm.kappa * cp) + s_shift[c];
                    double sw, cw;
                    sincospi(2.0 * ((double)(int32_t)r.beta * (1.0 / 4294967296.0)), &sw, &cw);
                    r.wr = (float)cw; r.wi = (float)sw;
                    r.flags = (fabs(sw) < 0.1) ? 1u : 0u;          // three-term recurrence ill-conditioned
                    r.mag = fabsf(g) * xi_mag;
                    r.b = b; r.e = e;
                    a.recs[(((size_t)c * n_pl + pl) * prm.n_tiles + tile) * prm.tile_cap + idx] = r;
                    my_bmin[c] = min(my_bmin[c], b);
                    my_bmax[c] = max(my_bmax[c], e);
                    int lo = max(b, 0), hi = min(e, prm.n_samples);
                    if (hi > lo) my_samples += (unsigned)(hi - lo);
                }
                if (kDebug) {
                    if (a.dbg_tau) a.dbg_tau[(size_t)c * F + f] = (rt + lr.r) / kC0;
                    if (a.dbg_grx) a.dbg_grx[(size_t)c * F + f] = grx_re;
                    if (a.dbg_amp) {
                        double turns = dR * prm.inv_lambda;
                        turns = (turns - floor(turns)) + a.carrier_frac_t0[p];
                        double sn, cn;
                        sincospi(-2.0 * turns, &sn, &cn);
                        double ar = (double)cg.x * xi.x - (double)cg.y * xi.y, ai = (double)cg.x * xi.y + (double)cg.y * xi.x;
                        a.dbg_amp[2 * ((size_t)c * F + f)] = ar * cn - ai * sn;
                        a.dbg_amp[2 * ((size_t)c * F + f) + 1] = ar * sn + ai * cn;
                    }
                }
            }
        }
    }
    // tile summaries
    for (int c = 0; c < C; ++c) {
        int lo = my_bmin[c], hi = my_bmax[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) { atomicMin(&s_bmin[c], lo); atomicMax(&s_bmax[c], hi); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) my_samples += __shfl_xor_sync(0xffffffffu, my_samples, o);
    if (lane == 0 && my_samples) atomicAdd(&s_samples, my_samples);
    __syncthreads();
    if (tid == 0) {
        a.tinfo[(size_t)pl * prm.n_tiles + tile].nrec = s_base;
        if (a.counters) {
            if (s_base) atomicAdd(a.counters + 0, (unsigned long long)s_base * C);
            if (s_samples) atomicAdd(a.counters + 1, s_samples);
        }
    }
    if (tid < C) {
        TileSpan sp;
        sp.bmin = s_bmin[tid]; sp.bmax_end = s_bmax[tid];
        sp.shift = s_shift[tid]; sp.pad = 0u;
        a.tspan[((size_t)tid * n_pl + pl) * prm.n_tiles + tile] = sp;
    }
}

}  // namespace

cudaError_t launch_geometry(const DevParams &prm, const GeometryArgs &a, int p0, int n_pl, cudaStream_t s)
{
    dim3 grid(prm.n_tiles, n_pl);
    const bool dbg = a.dbg_pos || a.dbg_tau || a.dbg_gtx || a.dbg_grx || a.dbg_amp || a.dbg_keep;
    if (dbg) geometry_kernel<true><<<grid, kThreads, 0, s>>>(prm, a, p0, n_pl);
    else     geometry_kernel<false><<<grid, kThreads, 0, s>>>(prm, a, p0, n_pl);
    return cudaGetLastError();
}

}  // namespace heeps
