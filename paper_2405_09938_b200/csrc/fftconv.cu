// K3s -- spectral echo accumulation: convolution of the range-slice moments with the waveform kernels
// (SURVEY.md §8(a) A6 "Moment/spectral" + A7; the range-sliced profile is "the impulse
// response of the surface and subsequently convolved by the waveform").
//
//   s_{c,p}[n] = exp(-j 2 pi f0 t0[p]) sum_{k<Kt} sum_{m<L} c_k[m] M_k[n - m]          (moments.cu header)
//
// One CTA = one (channel, pulse) vector.  The linear convolution is done as a circular one of length
// Nfft >= Ns + L - 1 in shared memory: Kt forward FFTs of the zero-padded moment rows, a multiply-accumulate
// with the precomputed spectra C_k (registers), one inverse FFT, the per-pulse reference phase, complex64
// store.  The FFT is an in-place radix-16 decimation-in-frequency network (register butterflies, twiddles
// from an fp64-built table); its digit-reversed output order is consumed as-is by the mirrored
// decimation-in-time inverse, and the C_k spectra are produced by the same forward code, so no reordering
// pass exists.  fp32 throughout: the transform's rounding (~1e-7 relative) is three orders under the
// 1e-4 parity budget.
//
// Bound: shared-memory bandwidth / FP32; HBM reads Kt moment rows and writes Ns samples per vector.
#include "kernels.cuh"

namespace heeps {

namespace {

constexpr int kKt = kMomentOrder;

__host__ __device__ constexpr int brev(int i, int bits)
{
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b);
    return r;
}
__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }

__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b)      // a * conj(b)
{
    return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y));
}

// exp(-2 pi i k / 16), k = 0..7
__device__ constexpr float kC16[8] = {1.f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f,
                                      0.f, -0.38268343236508977f, -0.70710678118654752f, -0.92387953251128674f};
__device__ constexpr float kS16[8] = {0.f, -0.38268343236508977f, -0.70710678118654752f, -0.92387953251128674f,
                                      -1.f, -0.92387953251128674f, -0.70710678118654752f, -0.38268343236508977f};

// R-point forward DFT in registers (radix-2 decimation in frequency): on return v[brev(r)] holds V[r].
template <int R>
__device__ __forceinline__ void dft_regs(float2 (&v)[R])
{
#pragma unroll
    for (int len = R; len >= 2; len >>= 1) {
#pragma unroll
        for (int st = 0; st < R; st += len) {
#pragma unroll
            for (int i = 0; i < len / 2; ++i) {
                const float2 a = v[st + i], b = v[st + i + len / 2];
                v[st + i] = make_float2(a.x + b.x, a.y + b.y);
                const float2 d = make_float2(a.x - b.x, a.y - b.y);
                const int k = i * (16 / len);
                if (k == 0) v[st + i + len / 2] = d;
                else if (k == 4) v[st + i + len / 2] = make_float2(d.y, -d.x);          // * (-i)
                else v[st + i + len / 2] = cmul(d, make_float2(kC16[k], kS16[k]));
            }
        }
    }
}

__device__ __forceinline__ int pad(int i) { return i + (i >> 4); }      // bank-conflict padding

// Twiddles w^r, r = 1..R-1, of one radix-R butterfly with base twiddle index j * tstep.  For R = 16 only w is loaded
// and the other fourteen are formed by complex products (w^2, w^4, w^8 by squaring): the FMA pipe idles while the L1 /
// shared-memory data path is what binds the kernel (profiles/r1_v11_k3s: l1tex 76 %), and the first pass's twiddles
// stride through the whole 64 KB table.  K3s 0.58 -> 0.36 ms on ATI; the angle error of w^8 is 8 roundings (~5e-7),
// parity unchanged (3.7e-6).
template <int R>
__device__ __forceinline__ void load_twiddles(float2 (&w)[R], const float2 *__restrict__ tw, int j, int tstep)
{
    if (R == 16) {
        w[1] = __ldg(tw + (size_t)j * tstep);
        w[2] = cmul(w[1], w[1]);
        w[4] = cmul(w[2], w[2]);
        w[8] = cmul(w[4], w[4]);
        w[3] = cmul(w[1], w[2]); w[5] = cmul(w[1], w[4]); w[6] = cmul(w[2], w[4]); w[7] = cmul(w[3], w[4]);
#pragma unroll
        for (int r = 9; r < 16; ++r) w[r < R ? r : 0] = cmul(w[(r - 8) < R ? (r - 8) : 0], w[8 < R ? 8 : 0]);
    } else {
#pragma unroll
        for (int r = 1; r < R; ++r) w[r] = __ldg(tw + (size_t)(j * r) * tstep);
    }
}

// One decimation-in-frequency pass: sub-transforms of size n_cur split into R of size n_cur / R.
template <int NFFT, int R, int THREADS>
__device__ __forceinline__ void fwd_pass(float2 *x, int n_cur, const float2 *__restrict__ tw)
{
    constexpr int bits = ilog2(R);
    const int s = n_cur / R, ls = 31 - __clz(s), tstep = NFFT / n_cur;
    for (int t = threadIdx.x; t < NFFT / R; t += THREADS) {
        const int j = t & (s - 1), base = (t >> ls) * n_cur + j;
        float2 v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = x[pad(base + q * s)];
        dft_regs<R>(v);
        float2 w[R];
        load_twiddles<R>(w, tw, j, tstep);
        x[pad(base)] = v[0];
#pragma unroll
        for (int r = 1; r < R; ++r) x[pad(base + r * s)] = cmul(v[brev(r, bits)], w[r]);
    }
    __syncthreads();
}

// The mirrored decimation-in-time pass (inverse transform, unnormalised).
template <int NFFT, int R, int THREADS>
__device__ __forceinline__ void inv_pass(float2 *x, int n_cur, const float2 *__restrict__ tw)
{
    constexpr int bits = ilog2(R);
    const int s = n_cur / R, ls = 31 - __clz(s), tstep = NFFT / n_cur;
    for (int t = threadIdx.x; t < NFFT / R; t += THREADS) {
        const int j = t & (s - 1), base = (t >> ls) * n_cur + j;
        float2 v[R], w[R];
        load_twiddles<R>(w, tw, j, tstep);
        v[0] = x[pad(base)];
        v[0].y = -v[0].y;
#pragma unroll
        for (int r = 1; r < R; ++r) {
            const float2 u = cmulc(x[pad(base + r * s)], w[r]);
            v[r] = make_float2(u.x, -u.y);                  // conj: IDFT(V) = conj(DFT(conj(V)))
        }
        dft_regs<R>(v);
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const float2 u = v[brev(q, bits)];
            x[pad(base + q * s)] = make_float2(u.x, -u.y);
        }
    }
    __syncthreads();
}

template <int NFFT, int THREADS>
__device__ __forceinline__ void fft_forward(float2 *x, const float2 *tw)
{
    constexpr int LOG = ilog2(NFFT), REM = 1 << (LOG % 4);
    int n_cur = NFFT;
#pragma unroll
    for (int k = 0; k < LOG / 4; ++k) { fwd_pass<NFFT, 16, THREADS>(x, n_cur, tw); n_cur >>= 4; }
    if (REM > 1) fwd_pass<NFFT, (REM > 1 ? REM : 2), THREADS>(x, n_cur, tw);
}

template <int NFFT, int THREADS>
__device__ __forceinline__ void fft_inverse(float2 *x, const float2 *tw)
{
    constexpr int LOG = ilog2(NFFT), REM = 1 << (LOG % 4);
    int n_cur = REM;
    if (REM > 1) inv_pass<NFFT, (REM > 1 ? REM : 2), THREADS>(x, n_cur, tw);
#pragma unroll
    for (int k = 0; k < LOG / 4; ++k) { n_cur <<= 4; inv_pass<NFFT, 16, THREADS>(x, n_cur, tw); }
}

template <int NFFT>
struct FftShape {
    static constexpr int kThreads = NFFT / 16 < 64 ? 64 : (NFFT / 16 > 512 ? 512 : NFFT / 16);
    static constexpr int kPerThread = NFFT / kThreads;
    static constexpr size_t kSmem = (size_t)(NFFT + NFFT / 16 + 1) * sizeof(float2);
};

template <int NFFT>
__global__ void __launch_bounds__(FftShape<NFFT>::kThreads)
fftconv_kernel(FftConvArgs a, int p0, int n_pl, int n_samples)
{
    constexpr int T = FftShape<NFFT>::kThreads, E = FftShape<NFFT>::kPerThread;
    extern __shared__ __align__(16) float2 xs[];
    const int pl = blockIdx.x, c = blockIdx.y, tid = threadIdx.x;
    const float2 *rows = a.mom + ((size_t)(c * n_pl + pl) * kKt) * a.nb_pad;
    if (a.nfft2) {                                         // fftconv_band_kernel takes empty and narrow vectors
        const int lo = __ldg(a.band_lo + (c * n_pl + pl)), hi = __ldg(a.band_hi + (c * n_pl + pl));
        if (hi <= lo || hi - lo + a.replica - 1 <= a.nfft2) return;
    }

    float2 acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = make_float2(0.f, 0.f);

    for (int k = 0; k < kKt; ++k) {
        const float2 *row = rows + (size_t)k * a.nb_pad;
#pragma unroll 4
        for (int e = 0; e < E; ++e) {
            const int i = tid + e * T;
            xs[pad(i)] = (i < a.nb) ? __ldg(row + i) : make_float2(0.f, 0.f);
        }
        __syncthreads();
        fft_forward<NFFT, T>(xs, a.tw);
        const float2 *ck = a.cspec + (size_t)k * NFFT;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int i = tid + e * T;
            const float2 u = cmul(xs[pad(i)], __ldg(ck + i));
            acc[e].x += u.x; acc[e].y += u.y;
        }
        __syncthreads();
    }
#pragma unroll
    for (int e = 0; e < E; ++e) xs[pad(tid + e * T)] = acc[e];
    __syncthreads();
    fft_inverse<NFFT, T>(xs, a.tw);

    // out[n] = y[n + L - 1] * exp(-j 2 pi f0 t0[p])      (A7; reference phase R0 = c0 t0[p])
    const double2 qd = __ldg(a.carrier_p + p0 + pl);
    const float2 q = make_float2((float)qd.x, (float)qd.y);
    float2 *dst = a.out + ((size_t)c * a.n_out_pulses + a.out_pulse0 + pl) * n_samples;
    for (int n = tid; n < n_samples; n += T) dst[n] = cmul(xs[pad(n + a.replica - 1)], q);
}

// The same convolution on the vector's occupied band alone.  K2k records the slice range [lo, hi) its echoes fall in
// (a scene spans a fraction of the sampling window: 450 of 5295 slices on ATI); when hi - lo + L - 1 <= N2 the linear
// convolution of the band with the L-tap kernels fits an N2-point circular one, four to eight times less transform work
// and moment-row traffic than the NFFT-point transform of the whole row.  With M'[i] = M[i + lo + L - 1] and
// y' = sum_k c_k * M'_k:  out[n] = y'[n - lo] for 0 <= n - lo < hi - lo + L - 1, zero elsewhere.  Vectors with a wider
// band are left to fftconv_kernel (launched beside this one); empty vectors are zero-filled here.
template <int N2>
__global__ void __launch_bounds__(FftShape<N2>::kThreads)
fftconv_band_kernel(FftConvArgs a, int p0, int n_pl, int n_samples)
{
    constexpr int T = FftShape<N2>::kThreads, E = FftShape<N2>::kPerThread;
    extern __shared__ __align__(16) float2 xs[];
    const int pl = blockIdx.x, c = blockIdx.y, tid = threadIdx.x;
    const int lo = __ldg(a.band_lo + (c * n_pl + pl)), hi = __ldg(a.band_hi + (c * n_pl + pl));
    float2 *dst = a.out + ((size_t)c * a.n_out_pulses + a.out_pulse0 + pl) * n_samples;
    if (hi <= lo) {
        for (int n = tid; n < n_samples; n += T) dst[n] = make_float2(0.f, 0.f);
        return;
    }
    const int W = hi - lo, L = a.replica;
    if (W + L - 1 > N2) return;
    const float2 *rows = a.mom + ((size_t)(c * n_pl + pl) * kKt) * a.nb_pad + (lo + L - 1);

    float2 acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = make_float2(0.f, 0.f);
    for (int k = 0; k < kKt; ++k) {
        const float2 *row = rows + (size_t)k * a.nb_pad;
#pragma unroll 4
        for (int e = 0; e < E; ++e) {
            const int i = tid + e * T;
            xs[pad(i)] = (i < W) ? __ldg(row + i) : make_float2(0.f, 0.f);
        }
        __syncthreads();
        fft_forward<N2, T>(xs, a.tw2);
        const float2 *ck = a.cspec2 + (size_t)k * N2;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int i = tid + e * T;
            const float2 u = cmul(xs[pad(i)], __ldg(ck + i));
            acc[e].x += u.x; acc[e].y += u.y;
        }
        __syncthreads();
    }
#pragma unroll
    for (int e = 0; e < E; ++e) xs[pad(tid + e * T)] = acc[e];
    __syncthreads();
    fft_inverse<N2, T>(xs, a.tw2);

    const double2 qd = __ldg(a.carrier_p + p0 + pl);
    const float2 q = make_float2((float)qd.x, (float)qd.y);
    const unsigned n_out = (unsigned)(W + L - 1);
    for (int n = tid; n < n_samples; n += T) {
        const int i = n - lo;
        dst[n] = ((unsigned)i < n_out) ? cmul(xs[pad(i)], q) : make_float2(0.f, 0.f);
    }
}

// Spectra of the waveform kernels: cspec[k] = FFT(zero-padded c_k) / NFFT, in the forward pass's order.
template <int NFFT>
__global__ void __launch_bounds__(FftShape<NFFT>::kThreads)
kernel_spectra_kernel(const float2 *ck, int replica, const float2 *tw, float2 *cspec)
{
    constexpr int T = FftShape<NFFT>::kThreads, E = FftShape<NFFT>::kPerThread;
    extern __shared__ __align__(16) float2 xs[];
    const int k = blockIdx.x, tid = threadIdx.x;
    for (int e = 0; e < E; ++e) {
        const int i = tid + e * T;
        xs[pad(i)] = (i < replica) ? ck[(size_t)k * replica + i] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    fft_forward<NFFT, T>(xs, tw);
    const float sc = 1.0f / (float)NFFT;
    for (int e = 0; e < E; ++e) {
        const int i = tid + e * T;
        const float2 u = xs[pad(i)];
        cspec[(size_t)k * NFFT + i] = make_float2(u.x * sc, u.y * sc);
    }
}

template <int NFFT>
cudaError_t launch_conv(const FftConvArgs &a, int p0, int n_pl, int n_channels, int n_samples, cudaStream_t s)
{
    constexpr size_t smem = FftShape<NFFT>::kSmem;
    if (smem > 48 * 1024) {
        cudaError_t rc = cudaFuncSetAttribute(fftconv_kernel<NFFT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (rc != cudaSuccess) return rc;
    }
    fftconv_kernel<NFFT><<<dim3(n_pl, n_channels), FftShape<NFFT>::kThreads, smem, s>>>(a, p0, n_pl, n_samples);
    return cudaGetLastError();
}

template <int N2>
cudaError_t launch_conv_band(const FftConvArgs &a, int p0, int n_pl, int n_channels, int n_samples, cudaStream_t s)
{
    constexpr size_t smem = FftShape<N2>::kSmem;
    if (smem > 48 * 1024) {
        cudaError_t rc = cudaFuncSetAttribute(fftconv_band_kernel<N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (rc != cudaSuccess) return rc;
    }
    fftconv_band_kernel<N2><<<dim3(n_pl, n_channels), FftShape<N2>::kThreads, smem, s>>>(a, p0, n_pl, n_samples);
    return cudaGetLastError();
}

template <int NFFT>
cudaError_t launch_spec(const float2 *ck, int replica, const float2 *tw, float2 *cspec, cudaStream_t s)
{
    constexpr size_t smem = FftShape<NFFT>::kSmem;
    if (smem > 48 * 1024) {
        cudaError_t rc = cudaFuncSetAttribute(kernel_spectra_kernel<NFFT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (rc != cudaSuccess) return rc;
    }
    kernel_spectra_kernel<NFFT><<<kKt, FftShape<NFFT>::kThreads, smem, s>>>(ck, replica, tw, cspec);
    return cudaGetLastError();
}

}  // namespace

#define HEEPS_FFT_SIZES(X) X(256) X(512) X(1024) X(2048) X(4096) X(8192) X(16384)

cudaError_t launch_fftconv(const DevParams &prm, const FftConvArgs &a, int p0, int n_pl, cudaStream_t s)
{
    if (a.nfft2) {
        if (!a.band_lo || !a.band_hi || !a.cspec2 || !a.tw2 || a.nfft2 >= a.nfft) return cudaErrorInvalidValue;
        cudaError_t rc;
        switch (a.nfft2) {
#define HEEPS_CASE(N) case N: rc = launch_conv_band<N>(a, p0, n_pl, prm.n_channels, prm.n_samples, s); break;
            HEEPS_FFT_SIZES(HEEPS_CASE)
#undef HEEPS_CASE
            default: return cudaErrorInvalidValue;
        }
        if (rc != cudaSuccess) return rc;
    }
    switch (a.nfft) {
#define HEEPS_CASE(N) case N: return launch_conv<N>(a, p0, n_pl, prm.n_channels, prm.n_samples, s);
        HEEPS_FFT_SIZES(HEEPS_CASE)
#undef HEEPS_CASE
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_kernel_spectra(int nfft, const float2 *ck, int replica, const float2 *tw, float2 *cspec,
                                  cudaStream_t s)
{
    switch (nfft) {
#define HEEPS_CASE(N) case N: return launch_spec<N>(ck, replica, tw, cspec, s);
        HEEPS_FFT_SIZES(HEEPS_CASE)
#undef HEEPS_CASE
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace heeps

// ---------------------------------------------------------------------------------------------------------------------
// sim_echoes_to_iq_static (include/heeps_sim.h) -- K3s for ONE (channel, pulse) vector with every byte of device memory
// it needs besides the caller's inputs and output in a file-scope static array: the moment rows (the scratch the moment
// kernels fill and fftconv_kernel reads), the waveform taps c_k, their spectra, the twiddle table and the vector's
// phase factor.  For callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses that
// forbid it): the entry point enqueues kernels and one memset on the caller's stream and calls no cudaMalloc / cudaFree
// or allocating library routine; the only set-up is one cudaGetSymbolAddress per device.  fftconv_kernel and
// kernel_spectra_kernel are the kernels of the normal path, launched on the static array.
// Every call shares the array (it keeps the last call's contents; the rows are cleared at the start of every call):
// two calls that overlap on one GPU (different streams, or threads) race.  Every GPU that loads the library holds
// the array (kStaticFloat2 * 8 bytes = 1.38 MB) until exit.
// ---------------------------------------------------------------------------------------------------------------------
#include <algorithm>
#include <cmath>
#include <mutex>

#include "../../include/heeps_sim.h"

namespace heeps {

namespace {

constexpr int kStaticMaxFft = SIM_STATIC_MAX_SLICES;              // Ns + L - 1 <= this
constexpr int kStaticMaxReplica = SIM_STATIC_MAX_REPLICA;
// [Kt][kStaticMaxFft] moment rows | [Kt][kStaticMaxFft] spectra | [kStaticMaxFft] twiddles | [Kt][kStaticMaxReplica] taps |
// 2 float2 = one double2 phase factor
constexpr size_t kStaticRows = 0, kStaticSpec = (size_t)kKt * kStaticMaxFft, kStaticTw = 2 * (size_t)kKt * kStaticMaxFft,
                 kStaticTaps = kStaticTw + kStaticMaxFft, kStaticPhase = kStaticTaps + (size_t)kKt * kStaticMaxReplica,
                 kStaticFloat2 = kStaticPhase + 2;
static __device__ __align__(256) float2 g_static_scratch[kStaticFloat2];

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the device address is looked up once
// per device, with that device current.
std::mutex g_static_mutex;
float2 *g_static_ptr[64] = {};

// Twiddles exp(-2 pi i k / nfft), the taps c_k[m] (Chebyshev coefficients in y of the slice response
// exp(j 2 pi kappa (m + (y + 1)/2 - L/2)^2), 64-node Gauss-Chebyshev quadrature -- the formula of sim_create's
// chebyshev_kernels, evaluated here on the device in fp64 so that nothing is copied from host memory) and the phase.
__global__ void __launch_bounds__(256)
static_tables_kernel(float2 *scratch, int nfft, int replica, double kappa, double ph_re, double ph_im)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < nfft) {
        double sn, cs;
        sincospi(-2.0 * (double)t / (double)nfft, &sn, &cs);
        scratch[kStaticTw + t] = make_float2((float)cs, (float)sn);
    }
    if (t == 0) *reinterpret_cast<double2 *>(scratch + kStaticPhase) = make_double2(ph_re, ph_im);
    if (t < replica) {
        constexpr int NQ = 64;
        double ar[kKt], ai[kKt];
#pragma unroll
        for (int k = 0; k < kKt; ++k) ar[k] = ai[k] = 0.0;
        for (int j = 0; j < NQ; ++j) {
            const double th = (j + 0.5) / NQ;                               // in units of pi
            const double u = (double)t + 0.5 * (cospi(th) + 1.0) - 0.5 * (double)replica;
            double turns = kappa * u * u;
            turns -= floor(turns);
            double gs, gc;
            sincospi(2.0 * turns, &gs, &gc);
#pragma unroll
            for (int k = 0; k < kKt; ++k) {
                const double ck = cospi((double)k * th);
                ar[k] = fma(gc, ck, ar[k]); ai[k] = fma(gs, ck, ai[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < kKt; ++k) {
            const double sc = (k ? 2.0 : 1.0) / NQ;
            scratch[kStaticTaps + (size_t)k * replica + t] = make_float2((float)(ar[k] * sc), (float)(ai[k] * sc));
        }
    }
}

// Moment rows from the caller's echo list: M_k[b + L - 1] += w T_k(2 eps - 1) (moments.cu header), by atomics.
__global__ void __launch_bounds__(256)
static_moments_kernel(float2 *rows, int nb, int nb_pad, int replica, const int32_t *slice, const float *eps,
                      const float2 *weight, long long n)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const long long idx = (long long)slice[e] + replica - 1;
        if (idx < 0 || idx >= nb) continue;                                 // the echo's window misses [0, Ns): clipped
        const float2 w = weight[e];
        const float y = fmaf(2.f, eps[e], -1.f);
        float t0 = 1.f, t1 = y;
        atomicAdd(rows + idx, w);
        atomicAdd(rows + nb_pad + idx, make_float2(w.x * t1, w.y * t1));
        for (int k = 2; k < kKt; ++k) {
            const float t2 = 2.f * y * t1 - t0;
            atomicAdd(rows + (size_t)k * nb_pad + idx, make_float2(w.x * t2, w.y * t2));
            t0 = t1; t1 = t2;
        }
    }
}

template <int NFFT>
cudaError_t static_run(float2 *scr, int n_samples, int replica, double kappa, double ph_re, double ph_im,
                       const int32_t *slice, const float *eps, const float2 *weight, long long n, float2 *out, cudaStream_t s)
{
    const int nb = n_samples + replica - 1, nb_pad = (nb + 3) & ~3;
    cudaError_t rc = cudaMemsetAsync(scr + kStaticRows, 0, (size_t)kKt * nb_pad * sizeof(float2), s);    // rows start at zero
    if (rc != cudaSuccess) return rc;
    static_tables_kernel<<<(std::max(NFFT, replica) + 255) / 256, 256, 0, s>>>(scr, NFFT, replica, kappa, ph_re, ph_im);
    if ((rc = cudaGetLastError()) != cudaSuccess) return rc;
    if ((rc = launch_spec<NFFT>(scr + kStaticTaps, replica, scr + kStaticTw, scr + kStaticSpec, s)) != cudaSuccess) return rc;
    if (n > 0) {
        const int blocks = (int)std::min<long long>((n + 255) / 256, 148 * 8);
        static_moments_kernel<<<blocks, 256, 0, s>>>(scr + kStaticRows, nb, nb_pad, replica, slice, eps, weight, n);
        if ((rc = cudaGetLastError()) != cudaSuccess) return rc;
    }
    FftConvArgs a{};
    a.mom = scr + kStaticRows; a.cspec = scr + kStaticSpec; a.tw = scr + kStaticTw;
    a.carrier_p = reinterpret_cast<const double2 *>(scr + kStaticPhase);
    a.out = out; a.n_out_pulses = 1; a.out_pulse0 = 0;
    a.nfft = NFFT; a.nb = nb; a.nb_pad = nb_pad; a.replica = replica;
    return launch_conv<NFFT>(a, 0, 1, 1, n_samples, s);
}

}  // namespace

}  // namespace heeps

extern "C" int sim_echoes_to_iq_static(double chirp_rate_hz_per_s, double chirp_len_s, double fs_hz, int32_t n_samples,
                                       const int32_t *slice_dev, const float *eps_dev, const float *weight_dev,
                                       int64_t n_echoes, const double phase[2], void *iq_dev, int device, void *cuda_stream)
{
    using namespace heeps;
    if (!(fs_hz > 0) || !(chirp_len_s > 0) || !std::isfinite(chirp_rate_hz_per_s) || !std::isfinite(chirp_len_s) ||
        !std::isfinite(fs_hz) || n_samples < 1 || n_echoes < 0 || !iq_dev || !phase || !std::isfinite(phase[0]) ||
        !std::isfinite(phase[1]) || (n_echoes > 0 && (!slice_dev || !eps_dev || !weight_dev)))
        return SIM_EINVAL;
    const double len = chirp_len_s * fs_hz, len_round = std::nearbyint(len);
    if (!(std::fabs(len - len_round) < 1e-9 * std::max(1.0, len)) || len_round < 1.0) return SIM_EINVAL;   // T fs integer
    const int replica = (int)len_round;
    // beyond the static array: a clear error, never a silent overrun
    if (replica > kStaticMaxReplica || (long long)n_samples + replica - 1 > kStaticMaxFft) return SIM_ERANGE;
    const double kappa = chirp_rate_hz_per_s / (2.0 * fs_hz * fs_hz);
    {   // Kt = 8 moments must resolve the chirp (Jacobi-Anger tail; sim_create applies the same bar to its taps)
        const double z = M_PI * std::fabs(kappa) * len;
        double tail = 0;
        for (int k = kKt; k < kKt + 4; ++k) tail += 2.0 * std::fabs(jn(k, z));
        if (!(tail <= 5e-6)) return SIM_EINVAL;
    }
    if (device < 0 || device >= 64) return SIM_EINVAL;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return SIM_ECUDA; }
    if (prev != device && cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return SIM_ECUDA; }
    float2 *scr = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_ptr[device]) {
            float2 *p = nullptr;
            if (cudaGetSymbolAddress((void **)&p, g_static_scratch) != cudaSuccess || !p) {
                cudaGetLastError();
                if (prev != device) cudaSetDevice(prev);
                return SIM_ECUDA;
            }
            g_static_ptr[device] = p;
        }
        scr = g_static_ptr[device];
    }
    int nfft = 256;
    while (nfft < n_samples + replica - 1) nfft <<= 1;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const float2 *w2 = reinterpret_cast<const float2 *>(weight_dev);
    float2 *out = static_cast<float2 *>(iq_dev);
    cudaError_t rc = cudaErrorInvalidValue;
    switch (nfft) {
#define HEEPS_CASE(N) case N: rc = static_run<N>(scr, n_samples, replica, kappa, phase[0], phase[1], slice_dev, eps_dev, w2, n_echoes, out, s); break;
        HEEPS_CASE(256) HEEPS_CASE(512) HEEPS_CASE(1024) HEEPS_CASE(2048) HEEPS_CASE(4096) HEEPS_CASE(8192)
#undef HEEPS_CASE
        default: break;
    }
    if (prev != device) cudaSetDevice(prev);
    if (rc != cudaSuccess) { cudaGetLastError(); return SIM_ECUDA; }
    return SIM_OK;
}
