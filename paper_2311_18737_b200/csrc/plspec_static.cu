// plspec_static.cu -- plspec_profile_static: the per-gate products of plspec_profile (include/plspec.h; SURVEY.md 8(f)
// NEXT-2; PAPER.md:40-45 Eq. 1, :79 Eq. 8) through an entry point that ALLOCATES NOTHING -- for callers that cannot
// call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// It is the (gate, column tile) variant of the products kernels of plspec_finalize_products (plspec_fused.cuh:
// finalize_products_kernel / products_tail_kernel): the CTAs of a gate meet in a 32-byte workspace per gate -- the
// arg maxima as 64-bit keys (value bits << 32 | ~bin: S >= 0, so the float's bit pattern orders like its value and
// the lowest bin wins a tie) through atomicMax, the sum of the searched bins through a float64 atomicAdd, and an
// arrival counter; the last CTA of a gate to arrive takes the bins near the lines out of the sum again and writes the
// five numbers.  There that workspace is cudaMalloc'ed per handle; HERE it is a file-scope array in device memory,
// g_profile_work below, of kStaticMaxGates entries (256 KiB, held by every GPU that loads the library until exit).
//
// In host code the array's name is a host-side stand-in, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, asked once per device with that device current (work_address below) and passed to the kernel.
//
// Every call shares the array and it keeps the last call's contents: each call first clears the entries it uses
// (cudaMemsetAsync on the caller's stream, ahead of the kernel).  Calls that overlap on the GPU (different streams,
// or different host threads on different streams) RACE on it; calls on one stream, or ordered by events, do not.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/plspec.h"

namespace {

constexpr int kStaticMaxGates = PLSPEC_STATIC_MAX_GATES;
constexpr int kTileBins = 4096;                 // bins of one row a CTA reads: 256 threads x 4 loads of 128 bits
constexpr int kMaxDevices = 64;

struct ProfileWork { unsigned long long up, dn; double sum; unsigned int arrived, pad; };
static_assert(sizeof(ProfileWork) == 32, "workspace entry is 32 bytes");

static __device__ __align__(256) ProfileWork g_profile_work[kStaticMaxGates];

// grid (tiles per row, gates); definitions of the five outputs: profile_kernel (plspec_kernels.cuh) / include/plspec.h
__global__ void __launch_bounds__(256) profile_tiles_kernel(const float *__restrict__ S, int N, int n_ipp, int k_min, int guard,
                                                            ProfileWork *__restrict__ work, int *__restrict__ k_up,
                                                            float *__restrict__ p_up, int *__restrict__ k_dn,
                                                            float *__restrict__ p_dn, float *__restrict__ noise) {
    __shared__ unsigned long long sb[2][8];
    __shared__ double ssum[8];
    __shared__ int scnt[8];
    __shared__ int s_last;
    const int gate = blockIdx.y;
    const float *row = S + (long long)gate * N;
    const float4 *row4 = reinterpret_cast<const float4 *>(row);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lo = k_min, hi = N - k_min, mid = N / 2;
    const int v0 = blockIdx.x * (kTileBins / 4), v1 = min(N / 4, v0 + kTileBins / 4);
    float4 v[4];
#pragma unroll
    for (int u = 0; u < 4; u++) {
        const int i = v0 + tid + u * 256;
        v[u] = i < v1 ? __ldg(row4 + i) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    unsigned long long up = 0, dn = 0;          // key 0 = "no bin": below every real key
    // a thread meets at most 16 bins: their sum in float32 (<= 15 roundings of 2^-24 relative, against the 1e-6 the
    // noise floor is good to), everything above in float64
    float facc = 0.f;
    auto take = [&](float x, int f) {
        if (f >= lo && f <= hi && f != mid) {
            const unsigned long long key = ((unsigned long long)__float_as_uint(x) << 32) | (unsigned)(~f);
            if (f < mid) up = key > up ? key : up; else dn = key > dn ? key : dn;
            facc += x;
        }
    };
#pragma unroll
    for (int u = 0; u < 4; u++) {
        const int i = v0 + tid + u * 256;
        if (i >= v1) continue;
        take(v[u].x, 4 * i); take(v[u].y, 4 * i + 1); take(v[u].z, 4 * i + 2); take(v[u].w, 4 * i + 3);
    }
    double acc = (double)facc;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        const unsigned long long u = __shfl_xor_sync(0xffffffffu, up, o), d = __shfl_xor_sync(0xffffffffu, dn, o);
        up = u > up ? u : up; dn = d > dn ? d : dn;
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
    }
    if (lane == 0) { sb[0][warp] = up; sb[1][warp] = dn; ssum[warp] = acc; }
    __syncthreads();
    ProfileWork *w = work + gate;
    if (tid == 0) {
        for (int k = 1; k < 8; k++) {
            up = sb[0][k] > up ? sb[0][k] : up; dn = sb[1][k] > dn ? sb[1][k] : dn;
            acc += ssum[k];
        }
        if (up) atomicMax(&w->up, up);
        if (dn) atomicMax(&w->dn, dn);
        atomicAdd(&w->sum, acc);
        __threadfence();                        // this CTA's three updates before its arrival
        s_last = atomicAdd(&w->arrived, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    // the last CTA of the gate: every other CTA's updates are ordered before its arrival, and the arrivals before ours
    __threadfence();
    const unsigned long long wu = *reinterpret_cast<volatile unsigned long long *>(&w->up);
    const unsigned long long wd = *reinterpret_cast<volatile unsigned long long *>(&w->dn);
    const double wsum = *reinterpret_cast<volatile double *>(&w->sum);
    const int ku = (int)~(unsigned)(wu & 0xffffffffu), kd = (int)~(unsigned)(wd & 0xffffffffu);
    // the bins within `guard` of either line (each once, inside the searched range): at most 2 (2 guard + 1)
    const int g = guard < N ? guard : N, wlen = 2 * g + 1;
    double ex = 0.0;
    int nex = 0;
    for (int j = tid; j < 2 * wlen; j += 256) {
        const bool second = j >= wlen;
        const int f = (second ? kd : ku) - g + (second ? j - wlen : j);
        const int du = f > ku ? f - ku : ku - f;
        if (f >= lo && f <= hi && f != mid && !(second && du <= g)) { ex += (double)row[f]; nex++; }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        ex += __shfl_xor_sync(0xffffffffu, ex, o);
        nex += __shfl_xor_sync(0xffffffffu, nex, o);
    }
    if (lane == 0) { ssum[warp] = ex; scnt[warp] = nex; }
    __syncthreads();
    if (tid == 0) {
        for (int k = 1; k < 8; k++) { ex += ssum[k]; nex += scnt[k]; }
        k_up[gate] = ku; k_dn[gate] = kd;
        p_up[gate] = __uint_as_float((unsigned)(wu >> 32)) / (float)n_ipp;
        p_dn[gate] = __uint_as_float((unsigned)(wd >> 32)) / (float)n_ipp;
        const int cnt = (hi - lo) - nex;        // hi - lo + 1 searched bins less N/2
        noise[gate] = cnt > 0 ? (float)((wsum - ex) / (double)cnt / (double)n_ipp) : 0.f;
    }
}

// Device address of g_profile_work on the current device: asked once per device, with that device current.
std::mutex g_mu;
ProfileWork *g_work_addr[kMaxDevices];          // zero-initialised; guarded by g_mu

int work_address(ProfileWork **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return PLSPEC_ERR_CUDA; }
    if (dev < 0 || dev >= kMaxDevices) return PLSPEC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_work_addr[dev]) {
        cudaDeviceProp prop;
        if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { (void)cudaGetLastError(); return PLSPEC_ERR_CUDA; }
        if (prop.major != 10 || prop.minor != 0) return PLSPEC_ERR_UNSUPPORTED;      // the library holds sm_100a code only
        ProfileWork *p = nullptr;
        if (cudaGetSymbolAddress((void **)&p, g_profile_work) != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return PLSPEC_ERR_CUDA;
        }
        g_work_addr[dev] = p;
    }
    *out = g_work_addr[dev];
    return PLSPEC_OK;
}

}  // namespace

extern "C" int plspec_profile_static(const float *S, int n_ranges, int N, int n_ipp, int k_min, int guard, int *k_up,
                                     float *p_up, int *k_dn, float *p_dn, float *noise, void *stream_) {
    if (!S || !k_up || !p_up || !k_dn || !p_dn || !noise) return PLSPEC_ERR_INVALID_ARG;
    if (N < 16 || N > 65536 || (N & (N - 1)) || n_ranges < 1 || n_ipp < 1 || k_min < 1 || k_min >= N / 2 || guard < 0)
        return PLSPEC_ERR_INVALID_ARG;
    if (n_ranges > kStaticMaxGates) return PLSPEC_ERR_INVALID_ARG;    // beyond the static workspace: use plspec_profile
    if ((uintptr_t)S & 15) return PLSPEC_ERR_INVALID_ARG;             // rows are read in 128-bit loads
    const void *ptrs[] = {S, k_up, p_up, k_dn, p_dn, noise};
    for (const void *p : ptrs) {                                      // device (or managed) memory only
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return PLSPEC_ERR_CUDA; }
        if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged) return PLSPEC_ERR_INVALID_ARG;
    }
    ProfileWork *work = nullptr;
    const int rc = work_address(&work);
    if (rc != PLSPEC_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    // the array keeps the last call's contents: maxima, sum and arrival counter of the entries used start at zero
    if (cudaMemsetAsync(work, 0, sizeof(ProfileWork) * (size_t)n_ranges, stream) != cudaSuccess) {
        (void)cudaGetLastError();
        return PLSPEC_ERR_CUDA;
    }
    const dim3 grid((unsigned)((N + kTileBins - 1) / kTileBins), (unsigned)n_ranges);
    profile_tiles_kernel<<<grid, 256, 0, stream>>>(S, N, n_ipp, k_min, guard, work, k_up, p_up, k_dn, p_dn, noise);
    if (cudaGetLastError() != cudaSuccess) return PLSPEC_ERR_CUDA;
    return PLSPEC_OK;
}
