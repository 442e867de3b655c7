// cufft_pipeline.cu -- COMPARISON POINT, NOT THE PRODUCT: the paper's own device structure, as written in
// PAPER.md section 3.2, on cuFFT.  Built into its own library (libplspec_cufft.so) so that libplspec.so never links
// cuFFT; only bench.py loads it (key `cufft_pipeline` of the bench line).
//
//   per pulse p (host loop, sec. 3.2.4):
//     K1 "complex multiplication": batch[r][t] = conj(TX[t]) * echo[r0 + r*step + t], one thread
//        per element of `batch` through a linearised index -> (r, t); zero for code_len <= t < N (reading A6)
//     K2 cuFFT: 1-D complex-to-complex FFT of every row of `batch`, in place, one plan
//        (cufftPlanMany) for the n_ranges rows
//     K3 "spectrum accumulation": spectrum[r][f] += |batch[r][f]|^2
//   `batch` (n_ranges x N complex) round-trips device memory between the three steps: that traffic
//   (>= 40 bytes per decoded sample) is what the fused kernel of libplspec.so removes.
//
// Differences from the paper's program, all in its favour: the inputs are already resident on the device (the
// paper copies one TX row and one echo row host -> device per pulse inside its timed region),
// 256-thread 1-D blocks instead of 16 x 16, and a bounds check instead of padding.
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <new>

namespace {

struct Ctx {
    int N, L, R, r0, stride, ipp_len, dtype;     // dtype: 0 = complex64 voltages, 1 = sc16 (int16 I, Q)
    cufftHandle plan;
    bool have_plan;
    float2 *batch;                               // [R][N], the paper's `batch` array
    long long launches;                          // kernels + cuFFT executions enqueued so far
};

__device__ __forceinline__ float2 load_echo(const void *V, long long i, int dtype) {
    if (dtype == 0) return reinterpret_cast<const float2 *>(V)[i];
    const short2 s = reinterpret_cast<const short2 *>(V)[i];
    return make_float2((float)s.x, (float)s.y);
}

// K1
__global__ void __launch_bounds__(256) complex_multiplication_kernel(const void *__restrict__ echo, const float2 *__restrict__ tx,
                                                                     float2 *__restrict__ batch, int N, int L, int R, int r0,
                                                                     int stride, int dtype) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)R * N) return;
    const int r = (int)(i / N), t = (int)(i - (long long)r * N);
    float2 d = make_float2(0.f, 0.f);
    if (t < L) {
        const float2 z = load_echo(echo, (long long)r0 + (long long)r * stride + t, dtype);
        const float2 c = tx[t];
        d = make_float2(z.x * c.x + z.y * c.y, z.y * c.x - z.x * c.y);      // z * conj(c)
    }
    batch[i] = d;
}

// K3
__global__ void __launch_bounds__(256) spectrum_accumulation_kernel(const float2 *__restrict__ batch, float *__restrict__ spectrum,
                                                                    long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float2 x = batch[i];
    spectrum[i] += x.x * x.x + x.y * x.y;
}

}  // namespace

extern "C" {

// returns 0 on success, -1 bad argument, -2 allocation, -3 CUDA / cuFFT failure
int plspec_cufft_create(int N, int code_len, int n_ranges, int r0, int stride, int ipp_len, int dtype, void **out) {
    if (!out) return -1;
    *out = nullptr;
    if (N < 2 || (N & (N - 1)) || code_len < 1 || code_len > N || n_ranges < 1 || r0 < 0 || stride < 1 ||
        (dtype != 0 && dtype != 1) || (long long)r0 + (long long)(n_ranges - 1) * stride + code_len > ipp_len)
        return -1;
    Ctx *c = new (std::nothrow) Ctx();
    if (!c) return -2;
    c->N = N; c->L = code_len; c->R = n_ranges; c->r0 = r0; c->stride = stride; c->ipp_len = ipp_len; c->dtype = dtype;
    c->have_plan = false; c->batch = nullptr; c->launches = 0;
    if (cudaMalloc((void **)&c->batch, sizeof(float2) * (size_t)n_ranges * (size_t)N) != cudaSuccess) {
        (void)cudaGetLastError();
        delete c;
        return -2;
    }
    int n[1] = {N};
    if (cufftPlanMany(&c->plan, 1, n, nullptr, 1, N, nullptr, 1, N, CUFFT_C2C, n_ranges) != CUFFT_SUCCESS) {
        cudaFree(c->batch);
        delete c;
        return -3;
    }
    c->have_plan = true;
    *out = c;
    return 0;
}

// spectrum[R][N] (device, natural bin order) += the n_ipp pulses; echo[n_ipp][ipp_len], tx[n_ipp][code_len] on the
// device.  Enqueues 3 n_ipp steps on `stream` and returns without synchronising.
int plspec_cufft_accumulate(void *ctx, const void *echo, const void *tx, int n_ipp, float *spectrum, void *stream_) {
    Ctx *c = static_cast<Ctx *>(ctx);
    if (!c || !echo || !tx || !spectrum || n_ipp < 0) return -1;
    cudaStream_t stream = (cudaStream_t)stream_;
    if (cufftSetStream(c->plan, stream) != CUFFT_SUCCESS) return -3;
    const long long n = (long long)c->R * c->N;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    const size_t esz = c->dtype == 0 ? 8 : 4;
    for (int p = 0; p < n_ipp; p++) {                                            // loop over the pulses
        const void *e = static_cast<const char *>(echo) + (size_t)p * (size_t)c->ipp_len * esz;
        const float2 *t = static_cast<const float2 *>(tx) + (size_t)p * (size_t)c->L;
        complex_multiplication_kernel<<<blocks, 256, 0, stream>>>(e, t, c->batch, c->N, c->L, c->R, c->r0, c->stride, c->dtype);
        if (cufftExecC2C(c->plan, c->batch, c->batch, CUFFT_FORWARD) != CUFFT_SUCCESS) return -3;
        spectrum_accumulation_kernel<<<blocks, 256, 0, stream>>>(c->batch, spectrum, n);
        c->launches += 3;
    }
    if (cudaGetLastError() != cudaSuccess) return -3;
    return 0;
}

long long plspec_cufft_launches(void *ctx) { return ctx ? static_cast<Ctx *>(ctx)->launches : 0; }

int plspec_cufft_destroy(void *ctx) {
    Ctx *c = static_cast<Ctx *>(ctx);
    if (!c) return 0;
    (void)cudaDeviceSynchronize();
    if (c->have_plan) cufftDestroy(c->plan);
    if (c->batch) cudaFree(c->batch);
    delete c;
    return 0;
}

}  // extern "C"
