// plspec_kernels.cuh -- the CUDA kernels of the hot path.
//
//   fused_kernel<R3, Q, DT>   decode + FFT + |X|^2 + accumulate for Nk = 1024*R3 in
//                             {1024 .. 16384}, N = Q*Nk; one CTA per (gate, q, IPP chunk);
//                             the window lives in registers, passes exchange through shared
//                             memory, S accumulators stay in registers across the chunk's IPPs.
//   generic_kernel<DT>        any power-of-two Nk in [16, 16384]: shared-memory radix-2 DIF;
//                             slow but simple, used for small N and as a second GPU
//                             implementation to cross-check the fused one.
//   interleave_kernel         S_out[r][Q*k + q] = S_dev[r][q][k] for the outer radix Q > 1.
//
// Index algebra of the fused kernel (forward DFT, W_n = exp(-2 pi i / n)):
//   outer (Q > 1, decimation in frequency):  x_q[m] = (sum_j d[m + j Nk] W_Q^{jq}) W_N^{mq},
//                                            X[Q k + q] = DFT_Nk(x_q)[k]
//   inner, Nk = 32 * 32 * R3, M1 = 32 R3:    m = t1 M1 + t2 R3 + t3,  k = f1 + 32 f2 + 1024 f3
//     pass 1: A[f1][n']     = sum_t1 x[t1 M1 + n'] W_32^{t1 f1},  B = A W_Nk^{n' f1}   (n' = t2 R3 + t3)
//     pass 2: Cc[f1][f2][t3] = sum_t2 B[f1][t2 R3 + t3] W_32^{t2 f2}, D = Cc W_M1^{t3 f2}
//     pass 3: X[k]          = sum_t3 D[f1][f2][t3] W_R3^{t3 f3}
//   Shared-memory exchange layout: element (row a, f1) at a*33 + f1 (float2 units); rows are
//   n' after pass 1 and f2 R3 + t3 after pass 2 (written in place).  From pass 2 on, lane == f1,
//   so every shared access and the final S update are contiguous across the warp.
#pragma once
#include "plspec_common.cuh"

namespace plspec {

// ------------------------------------------------------------------------------------------
// decode + outer radix-Q butterfly for one inner index m (zero-pad reading A6)
template <int Q, int DT>
__device__ __forceinline__ float2 load_decoded(const KParams &P, const void *Vrow, long long voff,
                                               const float2 *Crow, int m, int q) {
    float2 d[Q];
#pragma unroll
    for (int j = 0; j < Q; j++) {
        int t = m + j * P.Nk;
        if (t < P.L) {
            float2 z = load_voltage<DT>(Vrow, voff + t);
            float2 c = __ldg(Crow + t);
            d[j] = cmul_conj(z, c);
        } else {
            d[j] = make_float2(0.f, 0.f);
        }
    }
    if constexpr (Q == 1) {
        return d[0];
    } else {
        float2 x;
        if constexpr (Q == 2) {
            x = (q == 0) ? cadd(d[0], d[1]) : csub(d[0], d[1]);
        } else {
            static_assert(Q == 4, "outer radix must be 1, 2 or 4");
            // sum_j d[j] (-i)^{jq} = (d0 + (-1)^q d2) + (-i)^q (d1 + (-1)^q d3)
            float2 e, o;
            if (q & 1) { e = csub(d[0], d[2]); o = csub(d[1], d[3]); }
            else       { e = cadd(d[0], d[2]); o = cadd(d[1], d[3]); }
            if (q == 0)      x = cadd(e, o);
            else if (q == 1) x = make_float2(e.x + o.y, e.y - o.x);   // e - i o
            else if (q == 2) x = csub(e, o);
            else             x = make_float2(e.x - o.y, e.y + o.x);   // e + i o
        }
        if (q != 0) x = cmul(x, __ldg(P.twN + ((m * q) & (P.N - 1))));
        return x;
    }
}

__device__ __forceinline__ void tile_of_block(const KParams &P, int &r, int &q, int &p_begin, int &p_end) {
    int tile = blockIdx.x;
    r = tile % P.R;
    int rest = tile / P.R;
    q = rest % P.Q;
    int chunk = rest / P.Q;
    p_begin = (int)(((long long)chunk * P.n_ipp) / P.n_chunks);
    p_end = (int)(((long long)(chunk + 1) * P.n_ipp) / P.n_chunks);
}

// warp-uniform pass-2 twiddles W_{32 R3}^{t3 f2}, [t3][f2], for R3 = 2,4,8,16 back to back
// (offsets 0, 64, 192, 448; 960 entries).  Filled once per device by the host (plspec_api.cu).
__constant__ float2 c_tw2[960];
__host__ __device__ constexpr int tw2_offset(int R3) { return 32 * (R3 - 2); }

// ------------------------------------------------------------------------------------------
template <int R3, int Q, int DT>
__global__ void __launch_bounds__(32 * R3, 16 / R3) fused_kernel(const KParams P) {
    constexpr int M1 = 32 * R3;          // threads per CTA == rows of the exchange buffer
    constexpr int PITCH = 33;            // float2 units; 33 keeps lane-strided rows conflict-free
    constexpr int G = 32 / R3;           // pass-3 groups (values of f2) per thread
    extern __shared__ float2 sm[];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int r, q, p_begin, p_end;
    tile_of_block(P, r, q, p_begin, p_end);

    float acc[32];
#pragma unroll
    for (int i = 0; i < 32; i++) acc[i] = 0.f;

    const long long gate_off = (long long)P.r0 + (long long)r * P.stride;

    for (int p = p_begin; p < p_end; p++) {
        const float2 *Crow = P.C + (long long)p * P.L;
        const long long voff = (long long)p * P.v_pitch + gate_off;
        float2 v[32];
        // ---- pass 1: thread <-> n' = tid; inputs x[t1 M1 + tid], coalesced over the warp
#pragma unroll
        for (int t1 = 0; t1 < 32; t1++) v[t1] = load_decoded<Q, DT>(P, P.V, voff, Crow, t1 * M1 + tid, q);
        dft_dif<32>(v);                                           // v[j] = A[f1 = brev5(j)][tid]
        sfor<1, 32>([&](auto j_) {
            constexpr int j = decltype(j_)::value;
            constexpr int f1 = brev<5>(j);
            v[j] = cmul(v[j], __ldg(P.tw1 + f1 * M1 + tid));      // B = A W_Nk^{n' f1}
        });
        __syncthreads();                                          // previous window's readers are done
        sfor<0, 32>([&](auto j_) {
            constexpr int j = decltype(j_)::value;
            sm[tid * PITCH + brev<5>(j)] = v[j];
        });
        __syncthreads();
        // ---- pass 2: thread <-> (f1 = lane, t3 = warp); DFT over t2
#pragma unroll
        for (int t2 = 0; t2 < 32; t2++) v[t2] = sm[(t2 * R3 + warp) * PITCH + lane];
        dft_dif<32>(v);                                           // v[j] = Cc[f2 = brev5(j)]
        if constexpr (R3 == 1) {
            // Nk = 1024: done. X[f1 + 32 f2] = v[brev5^-1(f2)]
#pragma unroll
            for (int j = 0; j < 32; j++) acc[j] += v[j].x * v[j].x + v[j].y * v[j].y;
        } else {
            if (warp != 0) {
                sfor<1, 32>([&](auto j_) {
                    constexpr int j = decltype(j_)::value;
                    constexpr int f2 = brev<5>(j);
                    v[j] = cmul(v[j], c_tw2[tw2_offset(R3) + warp * 32 + f2]);   // D = Cc W_M1^{t3 f2}
                });
            }
            sfor<0, 32>([&](auto j_) {                           // in place: same slots this thread read
                constexpr int j = decltype(j_)::value;
                sm[(brev<5>(j) * R3 + warp) * PITCH + lane] = v[j];
            });
            __syncthreads();
            // ---- pass 3: thread <-> (f1 = lane, f2 = warp*G + g); DFT over t3; |X|^2; accumulate
#pragma unroll
            for (int g = 0; g < G; g++) {
                const int f2 = warp * G + g;
                float2 u[R3];
#pragma unroll
                for (int t3 = 0; t3 < R3; t3++) u[t3] = sm[(f2 * R3 + t3) * PITCH + lane];
                dft_dif<R3>(u);                                   // u[j] = X[f3 = brev(j)]
#pragma unroll
                for (int j = 0; j < R3; j++) acc[g * R3 + j] += u[j].x * u[j].x + u[j].y * u[j].y;
            }
        }
    }

    // ---- flush: S[r][q][k], k = f1 + 32 f2 + 1024 f3; 32 lanes = 32 consecutive floats
    float *Srow = P.S + ((long long)r * P.Q + q) * P.Nk;
    if constexpr (R3 == 1) {
        sfor<0, 32>([&](auto j_) {
            constexpr int j = decltype(j_)::value;
            float *dst = Srow + lane + 32 * brev<5>(j);
            if (P.use_atomic) atomicAdd(dst, acc[j]); else *dst += acc[j];
        });
    } else {
        constexpr int L3 = ilog2(R3);
#pragma unroll
        for (int g = 0; g < G; g++) {
            const int f2 = warp * G + g;
            sfor<0, R3>([&](auto j_) {
                constexpr int j = decltype(j_)::value;
                float *dst = Srow + lane + 32 * f2 + 1024 * brev<L3>(j);
                if (P.use_atomic) atomicAdd(dst, acc[g * R3 + j]); else *dst += acc[g * R3 + j];
            });
        }
    }
}

// ------------------------------------------------------------------------------------------
// Generic path: Nk complex samples + Nk accumulators in shared memory, radix-2 DIF, any
// power-of-two Nk in [16, 16384].  Twiddles come from the full-circle table twN.
template <int DT>
__global__ void generic_kernel(const KParams P) {
    extern __shared__ float2 gsm[];
    float2 *x = gsm;
    float *acc = reinterpret_cast<float *>(gsm + P.Nk);
    const int tid = threadIdx.x, T = blockDim.x, Nk = P.Nk;
    int r, q, p_begin, p_end;
    tile_of_block(P, r, q, p_begin, p_end);
    for (int i = tid; i < Nk; i += T) acc[i] = 0.f;
    const long long gate_off = (long long)P.r0 + (long long)r * P.stride;
    const int tw_step = P.N / Nk;                 // W_Nk^e = twN[e * tw_step]

    for (int p = p_begin; p < p_end; p++) {
        const float2 *Crow = P.C + (long long)p * P.L;
        const long long voff = (long long)p * P.v_pitch + gate_off;
        for (int m = tid; m < Nk; m += T) {
            float2 s = make_float2(0.f, 0.f);
            for (int j = 0; j < P.Q; j++) {       // outer radix: sum_j d[m + j Nk] W_Q^{jq}
                int t = m + j * Nk;
                if (t < P.L) {
                    float2 d = cmul_conj(load_voltage<DT>(P.V, voff + t), __ldg(Crow + t));
                    int e = (j * q) & (P.Q - 1);  // W_Q^e = twN[e N / Q]
                    if (e) d = cmul(d, __ldg(P.twN + e * (P.N / P.Q)));
                    s = cadd(s, d);
                }
            }
            if (q) s = cmul(s, __ldg(P.twN + ((m * q) & (P.N - 1))));
            x[m] = s;
        }
        __syncthreads();
        for (int half = Nk >> 1; half >= 1; half >>= 1) {
            const int wstep = (Nk / (2 * half)) * tw_step;
            for (int b = tid; b < (Nk >> 1); b += T) {
                int k = b & (half - 1);
                int i = ((b - k) << 1) + k;
                float2 a = x[i], c = x[i + half];
                x[i] = cadd(a, c);
                float2 d = csub(a, c);
                x[i + half] = k ? cmul(d, __ldg(P.twN + k * wstep)) : d;
            }
            __syncthreads();
        }
        for (int i = tid; i < Nk; i += T) acc[i] += x[i].x * x[i].x + x[i].y * x[i].y;
        // next iteration rewrites x[m] with m == i (mod T): same thread, no barrier needed
    }
    float *Srow = P.S + ((long long)r * P.Q + q) * Nk;
    const int sh = 32 - P.log2Nk;
    for (int i = tid; i < Nk; i += T) {
        int k = (int)(__brev((unsigned)i) >> sh);      // DIF leaves X[brev(i)] at position i
        if (P.use_atomic) atomicAdd(Srow + k, acc[i]); else Srow[k] += acc[i];
    }
}

// S_out[r][Q k + q] = S_dev[r][q][k]
__global__ void interleave_kernel(const float *__restrict__ Sdev, float *__restrict__ Sout,
                                  int Q, int Nk, long long total) {
    const int N = Q * Nk;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        long long r = i / N;
        int f = (int)(i - r * N);
        int q = f % Q, k = f / Q;
        Sout[i] = Sdev[(r * Q + q) * Nk + k];
    }
}

}  // namespace plspec
