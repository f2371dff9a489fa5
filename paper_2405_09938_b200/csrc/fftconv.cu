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
