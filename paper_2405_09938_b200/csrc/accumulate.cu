// K3 -- echo accumulation, direct form ("the complex
// amplitudes of all facets lying in range slices ... are added to obtain one time sample",
// here with the chirp replica written out instead of a later convolution).
//
//   acc[c][p][n] += |A~_f| exp(j 2 pi (phi_f + beta_f (n - n_mid)))      for n in [b_f, e_f)
//
// (the facet-independent factor exp(j 2 pi kappa (n-n_mid)^2) is applied once per output sample
// in K4; arg A~ is folded into phi by K2).  After this dechirp every facet-echo is a windowed
// pure tone, so a thread that owns R CONSECUTIVE samples needs one sincos (MUFU) for its first
// sample and then advances by recurrence.  Two recurrences, chosen per record by K2:
//   * three-term  z[j+1] = 2cos(theta) z[j] - z[j-1]   -- one packed FFMA2 per sample; used when
//     |sin theta| >= 0.1, where the fp32 rounding of 2cos(theta) moves theta by < 6e-7 rad/sample;
//   * complex rotation z[j+1] = w z[j]                  -- 4 scalar ops; for theta near 0 or pi.
// The accumulate is one packed FADD2, so the hot loop is FADD2 + FFMA2 = 4 FP32 lane-operations
// and 2 issue slots per facet-sample (sm_100 f32x2 instructions).  The start phase is 32-bit fixed
// point (one IMAD, exact modulo one turn): no large floating-point phase is ever formed
// (SURVEY.md §7 hard part 5).
//
// Mapping: one CTA = (spatial tile, pulse, channel).  The tile's records (32 B each) are staged
// through shared memory and broadcast; warp k owns samples [lo + 32 R k, lo + 32 R (k+1)) of the
// tile's span [lo, hi) -- a spatial tile is narrow in delay, so span ~ L + a few tens of samples.
// Window edges are resolved per warp: a warp entirely inside [b, e) runs the unpredicated loop, an
// edge warp the predicated one, a warp outside skips the record.  Partial sums leave the CTA as
// fp64 atomics (RED.ADD.F64), once per CTA and sample.
//
// Bound: FP32 pipe, 4 lane-ops per facet-sample (+ ~12/R per-record set-up); XU 2/R.
#include "kernels.cuh"

namespace heeps {

namespace {

constexpr int kChunk = 256;          // records staged per shared-memory refill (8 KB)

// keep a loop invariant in a register: stops ptxas re-materialising it inside the record loop
__device__ __forceinline__ void pin(int &x) { asm volatile("" : "+r"(x)); }
__device__ __forceinline__ void pin(uint32_t &x) { asm volatile("" : "+r"(x)); }

template <int R>
__global__ void __launch_bounds__(512)
accumulate_kernel(DevParams prm, AccumulateArgs a, int n_pl)
{
    __shared__ uint4 s_rec[kChunk * 2];
    const int tile = blockIdx.x, pl = blockIdx.y, c = blockIdx.z;
    const int nrec = a.tinfo[(size_t)pl * prm.n_tiles + tile].nrec;
    if (nrec == 0) return;
    const size_t slot = ((size_t)c * n_pl + pl) * prm.n_tiles + tile;
    const TileSpan sp = a.tspan[slot];
    const int lo = max(sp.bmin, 0), hi = min(sp.bmax_end, prm.n_samples);
    if (hi <= lo) return;
    const uint4 *recs = reinterpret_cast<const uint4 *>(a.recs + slot * prm.tile_cap);
    double *out = reinterpret_cast<double *>(a.acc + ((size_t)c * n_pl + pl) * prm.n_samples);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int width = blockDim.x * R;

    for (int pass_lo = lo; pass_lo < hi; pass_lo += width) {
        int seg_lo = pass_lo + warp * 32 * R, seg_hi = seg_lo + 32 * R;
        int n0 = pass_lo + tid * R;
        const bool warp_active = seg_lo < hi;
        uint32_t k0 = (uint32_t)(n0 - prm.n_mid);
        pin(seg_lo); pin(seg_hi); pin(n0); pin(k0);
        float2 acc[R];
#pragma unroll
        for (int j = 0; j < R; ++j) acc[j] = make_float2(0.f, 0.f);

        for (int r0 = 0; r0 < nrec; r0 += kChunk) {
            const int nchunk = min(kChunk, nrec - r0);
            __syncthreads();
            for (int k = tid; k < nchunk * 2; k += blockDim.x) s_rec[k] = __ldg(recs + (size_t)r0 * 2 + k);
            __syncthreads();
            if (!warp_active) continue;
#pragma unroll 1
            for (int r = 0; r < nchunk; ++r) {
                const uint4 q1 = s_rec[2 * r + 1];                        // {wr, wi, b, e}
                const int b = (int)q1.z, e = (int)q1.w;
                if (seg_hi <= b || seg_lo >= e) continue;                 // warp-uniform: outside
                const uint4 q0 = s_rec[2 * r];                            // {phi, beta, |A|, flags}
                const uint32_t ph = q0.x + q0.y * k0;                     // turns * 2^32, exact mod 1
                const float t = __uint_as_float((ph >> 9) | 0x3f800000u) - 1.5f;   // [-0.5, 0.5) turns
                float sn, cs;
                __sincosf(t * 6.283185307179586f, &sn, &cs);
                const float mag = __uint_as_float(q0.z);
                const float wr = __uint_as_float(q1.x), wi = __uint_as_float(q1.y);
                float2 z0 = make_float2(mag * cs, mag * sn);
                float2 z1 = make_float2(z0.x * wr - z0.y * wi, z0.x * wi + z0.y * wr);
                const bool interior = seg_lo >= b && seg_hi <= e;         // warp-uniform
                if (q0.w == 0u) {                                         // three-term recurrence
                    const float c2 = wr + wr;
                    const float2 cc = make_float2(c2, c2);
                    if (interior) {
#pragma unroll
                        for (int j = 0; j < R; j += 2) {
                            acc[j] = __fadd2_rn(acc[j], z0);
                            if (j + 2 < R) z0 = __ffma2_rn(cc, z1, make_float2(-z0.x, -z0.y));
                            if (j + 1 < R) acc[j + 1] = __fadd2_rn(acc[j + 1], z1);
                            if (j + 3 < R) z1 = __ffma2_rn(cc, z0, make_float2(-z1.x, -z1.y));
                        }
                    } else {
                        const uint32_t cnt = (uint32_t)(e - b);
                        const int d0 = n0 - b;
#pragma unroll
                        for (int j = 0; j < R; j += 2) {
                            if ((uint32_t)(d0 + j) < cnt) acc[j] = __fadd2_rn(acc[j], z0);
                            if (j + 2 < R) z0 = __ffma2_rn(cc, z1, make_float2(-z0.x, -z0.y));
                            if (j + 1 < R && (uint32_t)(d0 + j + 1) < cnt) acc[j + 1] = __fadd2_rn(acc[j + 1], z1);
                            if (j + 3 < R) z1 = __ffma2_rn(cc, z0, make_float2(-z1.x, -z1.y));
                        }
                    }
                } else {                                                  // rotation (theta near 0 or pi)
                    const uint32_t cnt = (uint32_t)(e - b);
                    const int d0 = n0 - b;
#pragma unroll
                    for (int j = 0; j < R; ++j) {
                        if ((uint32_t)(d0 + j) < cnt) acc[j] = __fadd2_rn(acc[j], z0);
                        z0 = z1;
                        z1 = make_float2(z0.x * wr - z0.y * wi, z0.x * wi + z0.y * wr);
                    }
                }
            }
        }
        if (warp_active) {
#pragma unroll
            for (int j = 0; j < R; ++j) {
                const int n = n0 + j;
                if (n < hi) {
                    atomicAdd(out + 2 * (size_t)n, (double)acc[j].x);
                    atomicAdd(out + 2 * (size_t)n + 1, (double)acc[j].y);
                }
            }
        }
    }
}

}  // namespace

int accumulate_pick_r(double span_est)
{   // samples per thread: minimise (warp-quantised span) x (per-sample + per-record issue cost)
    const int cand[5] = {8, 10, 12, 14, 16};
    int best = 8;
    double best_cost = 1e300;
    for (int k = 0; k < 5; ++k) {
        const int r = cand[k];
        const double warps = ceil(span_est / (32.0 * r));
        const double cost = warps * 32.0 * (2.0 * r + 26.0);
        if (cost < best_cost) { best_cost = cost; best = r; }
    }
    return best;
}

cudaError_t launch_accumulate(const DevParams &prm, const AccumulateArgs &a, int n_pl, cudaStream_t s)
{
    dim3 grid(prm.n_tiles, n_pl, prm.n_channels);
    switch (a.samples_per_thread) {
        case 8:  accumulate_kernel<8><<<grid, a.block_threads, 0, s>>>(prm, a, n_pl); break;
        case 10: accumulate_kernel<10><<<grid, a.block_threads, 0, s>>>(prm, a, n_pl); break;
        case 12: accumulate_kernel<12><<<grid, a.block_threads, 0, s>>>(prm, a, n_pl); break;
        case 14: accumulate_kernel<14><<<grid, a.block_threads, 0, s>>>(prm, a, n_pl); break;
        case 16: accumulate_kernel<16><<<grid, a.block_threads, 0, s>>>(prm, a, n_pl); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace heeps
