// K3 -- echo accumulation, direct form ("the complex
// amplitudes of all facets lying in range slices ... are added to obtain one time sample",
// here with the chirp replica written out instead of a later convolution).
//
//   acc[c][p][n] += A~_f exp(j 2 pi (phi_f + beta_f (n - n_mid)))      for n in [b_f, b_f + cnt_f)
//
// (the facet-independent factor exp(j 2 pi kappa (n-n_mid)^2) is applied once per output sample
// in K4).  After the dechirp every facet-echo is a windowed pure tone, so a thread that owns R
// CONSECUTIVE samples needs one sincos (MUFU) for its first sample and then advances by the
// record's one-sample step w = exp(j 2 pi beta): 4 FP32 ops + 2 adds per facet-sample, no
// transcendental in the inner loop.  The start phase is 32-bit fixed point (one IMAD, exact
// modulo 1 turn), so no large floating-point phase is ever formed (SURVEY.md §7 hard part 5).
//
// Mapping: one CTA = (spatial tile, pulse, channel).  The tile's records (<= tile_cap, 32 B each)
// are staged through shared memory and broadcast; warp k owns samples
// [lo + 32 R k, lo + 32 R (k+1)) of the tile's span [lo, hi) -- a spatial tile is narrow in delay,
// so span ~ L + a few tens of samples.  Window edges are resolved per warp: a warp entirely
// inside [b, b+cnt) runs the unpredicated loop, an edge warp the predicated one, a warp
// outside skips the record.  Partial sums leave the CTA as fp64 atomics (RED.ADD.F64).
//
// Bound: FP32 pipe (6 FP32-pipe ops per facet-sample + ~14/R per-record overhead), XU 2/R.
#include "kernels.cuh"

namespace heeps {

namespace {

constexpr int kChunk = 256;          // records staged per shared-memory refill (8 KB)

template <int R>
__global__ void __launch_bounds__(1024)
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
        const int seg_lo = pass_lo + warp * 32 * R, seg_hi = seg_lo + 32 * R;
        const int n0 = pass_lo + tid * R;
        const bool warp_active = seg_lo < hi;
        const uint32_t k0 = (uint32_t)(n0 - prm.n_mid);
        float accr[R], acci[R];
#pragma unroll
        for (int j = 0; j < R; ++j) { accr[j] = 0.f; acci[j] = 0.f; }

        for (int r0 = 0; r0 < nrec; r0 += kChunk) {
            const int nchunk = min(kChunk, nrec - r0);
            __syncthreads();
            for (int k = tid; k < nchunk * 2; k += blockDim.x) s_rec[k] = __ldg(recs + (size_t)r0 * 2 + k);
            __syncthreads();
            if (!warp_active) continue;
            for (int r = 0; r < nchunk; ++r) {
                const uint4 q1 = s_rec[2 * r + 1];
                const int b = (int)q1.z, e = b + (int)q1.w;
                if (seg_hi <= b || seg_lo >= e) continue;                // warp-uniform
                const uint4 q0 = s_rec[2 * r];
                const uint32_t ph = q0.x + q0.y * k0;                    // turns * 2^32, exact mod 1
                const float t = __uint_as_float((ph >> 9) | 0x3f800000u) - 1.5f;   // [-0.5, 0.5) turns
                float sn, cs;
                __sincosf(t * 6.283185307179586f, &sn, &cs);
                const float ar = __uint_as_float(q0.z), ai = __uint_as_float(q0.w);
                const float wr = __uint_as_float(q1.x), wi = __uint_as_float(q1.y);
                float zr = ar * cs - ai * sn, zi = ar * sn + ai * cs;
                if (seg_lo >= b && seg_hi <= e) {                        // warp-uniform: interior
#pragma unroll
                    for (int j = 0; j < R; ++j) {
                        accr[j] += zr; acci[j] += zi;
                        const float tr = zr * wr - zi * wi;
                        zi = zr * wi + zi * wr;
                        zr = tr;
                    }
                } else {                                                 // edge warp: per-sample rect
                    const uint32_t cnt = q1.w;
                    const int d0 = n0 - b;
#pragma unroll
                    for (int j = 0; j < R; ++j) {
                        if ((uint32_t)(d0 + j) < cnt) { accr[j] += zr; acci[j] += zi; }
                        const float tr = zr * wr - zi * wi;
                        zi = zr * wi + zi * wr;
                        zr = tr;
                    }
                }
            }
        }
        if (warp_active) {
#pragma unroll
            for (int j = 0; j < R; ++j) {
                const int n = n0 + j;
                if (n < hi) {
                    atomicAdd(out + 2 * (size_t)n, (double)accr[j]);
                    atomicAdd(out + 2 * (size_t)n + 1, (double)acci[j]);
                }
            }
        }
    }
}

}  // namespace

cudaError_t launch_accumulate(const DevParams &prm, const AccumulateArgs &a, int n_pl, cudaStream_t s)
{
    dim3 grid(prm.n_tiles, n_pl, prm.n_channels);
    accumulate_kernel<8><<<grid, a.block_threads, 0, s>>>(prm, a, n_pl);
    return cudaGetLastError();
}

}  // namespace heeps
