// Pipe-throughput microbenchmarks ("FP32/XU/FP64 pipe peaks are not measured
// [by the driver] -- the builder must microbenchmark them ... in the same run"): the roofline
// denominators of the ALU-bound kernels (K3 on the FP32 pipe, K1/K2 on the FP64 pipe).
//
// Each kernel keeps kChains independent dependency chains per thread busy with one instruction
// kind; the chip is filled with 148 x 8 CTAs of 256 threads.  The figure returned is LANE
// operations per second (a packed f32x2 instruction counts 2, an FMA counts 1 operation).
#include <cuda_runtime.h>

#include "../../include/heeps_sim.h"

namespace {

constexpr int kChains = 8;
constexpr int kIters = 2048;

enum Kind { kFfma = 0, kFfma2, kFadd2, kMixFfma2Fadd2, kMufuSinCos, kDfma, kFaddScalar, kKinds };

template <int KIND>
__global__ void __launch_bounds__(256) pipe_kernel(float seed, float *sink)
{
    const float a = seed + 1e-7f * threadIdx.x;
    if (KIND == kFfma) {
        float x[kChains];
#pragma unroll
        for (int k = 0; k < kChains; ++k) x[k] = a + k;
        for (int it = 0; it < kIters; ++it) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) x[k] = fmaf(x[k], a, seed);
        }
        float s = 0;
#pragma unroll
        for (int k = 0; k < kChains; ++k) s += x[k];
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == kFaddScalar) {
        float x[kChains];
#pragma unroll
        for (int k = 0; k < kChains; ++k) x[k] = a + k;
        for (int it = 0; it < kIters; ++it) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) x[k] = __fadd_rn(x[k], a);
        }
        float s = 0;
#pragma unroll
        for (int k = 0; k < kChains; ++k) s += x[k];
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == kFfma2 || KIND == kFadd2 || KIND == kMixFfma2Fadd2) {
        float2 x[kChains];
        const float2 m = make_float2(a, a * 0.5f), c = make_float2(seed, -seed);
#pragma unroll
        for (int k = 0; k < kChains; ++k) x[k] = make_float2(a + k, a - k);
        for (int it = 0; it < kIters; ++it) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) {
                if (KIND == kFfma2) x[k] = __ffma2_rn(x[k], m, c);
                else if (KIND == kFadd2) x[k] = __fadd2_rn(x[k], m);
                else x[k] = (k & 1) ? __ffma2_rn(x[k], m, c) : __fadd2_rn(x[k], m);
            }
        }
        float s = 0;
#pragma unroll
        for (int k = 0; k < kChains; ++k) s += x[k].x + x[k].y;
        if (s == 12345.678f) sink[0] = s;
    } else if (KIND == kMufuSinCos) {
        float x[kChains];
#pragma unroll
        for (int k = 0; k < kChains; ++k) x[k] = a + 0.1f * k;
        for (int it = 0; it < kIters; ++it) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) x[k] = (k & 1) ? __sinf(x[k]) : __cosf(x[k]);
        }
        float s = 0;
#pragma unroll
        for (int k = 0; k < kChains; ++k) s += x[k];
        if (s == 12345.678f) sink[0] = s;
    } else {
        double x[kChains];
        const double da = a, ds = seed;
#pragma unroll
        for (int k = 0; k < kChains; ++k) x[k] = da + k;
        for (int it = 0; it < kIters; ++it) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) x[k] = fma(x[k], da, ds);
        }
        double s = 0;
#pragma unroll
        for (int k = 0; k < kChains; ++k) s += x[k];
        if (s == 12345.678) sink[0] = (float)s;
    }
}

template <int KIND>
cudaError_t time_kind(int blocks, float *sink, double *ops_per_s)
{
    cudaEvent_t e0, e1;
    cudaError_t rc;
    if ((rc = cudaEventCreate(&e0)) != cudaSuccess) return rc;
    if ((rc = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return rc; }
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {      // first repetition doubles as warm-up
        cudaEventRecord(e0);
        pipe_kernel<KIND><<<blocks, 256>>>(0.999f, sink);
        cudaEventRecord(e1);
        rc = cudaEventSynchronize(e1);
        if (rc != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (rc != cudaSuccess) return rc;
    const double per_instr = (KIND == kFfma2 || KIND == kFadd2 || KIND == kMixFfma2Fadd2) ? 2.0 : 1.0;
    *ops_per_s = (double)blocks * 256.0 * kChains * kIters * per_instr / (best * 1e-3);
    return cudaGetLastError();
}

}  // namespace

extern "C" int sim_measure_pipe_peaks(int device, sim_pipe_peaks *out)
{
    if (!out) return SIM_EINVAL;
    int prev = -1, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return SIM_ECUDA; }
    cudaGetDevice(&prev);
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return SIM_ECUDA; }
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    const int blocks = sms * 8;
    float *sink = nullptr;
    cudaError_t rc = cudaMalloc(reinterpret_cast<void **>(&sink), sizeof(float));
    if (rc == cudaSuccess) rc = time_kind<kFfma>(blocks, sink, &out->ffma_per_s);
    if (rc == cudaSuccess) rc = time_kind<kFaddScalar>(blocks, sink, &out->fadd_per_s);
    if (rc == cudaSuccess) rc = time_kind<kFfma2>(blocks, sink, &out->ffma2_lane_per_s);
    if (rc == cudaSuccess) rc = time_kind<kFadd2>(blocks, sink, &out->fadd2_lane_per_s);
    if (rc == cudaSuccess) rc = time_kind<kMixFfma2Fadd2>(blocks, sink, &out->mix_f32x2_lane_per_s);
    if (rc == cudaSuccess) rc = time_kind<kMufuSinCos>(blocks, sink, &out->mufu_per_s);
    if (rc == cudaSuccess) rc = time_kind<kDfma>(blocks, sink, &out->dfma_per_s);
    out->sm_count = sms;
    if (sink) cudaFree(sink);
    if (prev >= 0) cudaSetDevice(prev);
    if (rc != cudaSuccess) { cudaGetLastError(); return SIM_ECUDA; }
    return SIM_OK;
}
