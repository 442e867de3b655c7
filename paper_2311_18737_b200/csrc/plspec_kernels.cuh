// plspec_kernels.cuh -- decode/load helper shared by both kernels, and the generic kernel.
//
//   load_decoded<Q, DT>     sc16 -> fp32 (a1), window addressing (a2), decode by conj(code) (a3) and the
//                           outer radix-Q decimation-in-frequency butterfly for N = Q * Nk > 16384:
//                             x_q[m] = (sum_j d[m + j Nk] W_Q^{jq}) W_N^{mq},   X[Q k + q] = DFT_Nk(x_q)[k]
//   generic_kernel<DT>      any power-of-two Nk in [16, 16384]: shared-memory radix-2 DIF; slow but simple,
//                           used for N < 1024 and as a second GPU implementation to cross-check the
//                           fused kernel (plspec_fused.cuh).
#pragma once
#include "plspec_common.cuh"

namespace plspec {

// ------------------------------------------------------------------------------------------
// decode + outer radix-Q butterfly for one inner index m (zero-pad reading A6)
// outer radix-Q decimation-in-frequency butterfly + twiddle W_N^{mq} on Q decoded samples d[j] = d(m + j Nk)
template <int Q>
__device__ __forceinline__ float2 outer_bfly(const KParams &P, const float2 (&d)[Q], int m, int q) {
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

// where one IPP's voltages come from: global memory (V + voff) or the CTA's shared-memory stage
// (element index sbase + t; filled by cp.async.bulk in the fused kernel, plspec_fused.cuh)
struct VSrc {
    const void *V;
    long long voff;
    const unsigned char *stage;
    int sbase;
};

template <int DT, bool STAGED>
__device__ __forceinline__ float2 fetch_voltage(const VSrc &s, int t) {
    if constexpr (STAGED) {
        if constexpr (DT == DT_CF32) return reinterpret_cast<const float2 *>(s.stage)[s.sbase + t];
        else return sc16_to_f32(reinterpret_cast<const uint32_t *>(s.stage)[s.sbase + t]);
    } else {
        return load_voltage<DT>(s.V, s.voff + t);
    }
}

template <int Q, int DT, bool STAGED = false>
__device__ __forceinline__ float2 load_decoded(const KParams &P, const VSrc &src, const float2 *Crow, int m, int q) {
    float2 d[Q];
#pragma unroll
    for (int j = 0; j < Q; j++) {
        int t = m + j * P.Nk;
        if (t < P.L) {
            float2 z = fetch_voltage<DT, STAGED>(src, t);
            float2 c = __ldg(Crow + t);
            d[j] = cmul_conj(z, c);
        } else {
            d[j] = make_float2(0.f, 0.f);
        }
    }
    return outer_bfly<Q>(P, d, m, q);
}

// BPSK fast path (code_len == N, every code sample exactly +-1 + 0j, found by pack_codes_kernel):
// decode = sign flip.  cw[j] holds this thread's code bits of outer block j, bit `BIT` = 1 for -1.
template <int Q, int DT, int BIT, bool STAGED = false>
__device__ __forceinline__ float2 load_decoded_bpsk(const KParams &P, const VSrc &src, const uint32_t (&cw)[Q],
                                                    int m, int q) {
    float2 d[Q];
#pragma unroll
    for (int j = 0; j < Q; j++) {
        float2 z = fetch_voltage<DT, STAGED>(src, m + j * P.Nk);
        const uint32_t s = (cw[j] << (31 - BIT)) & 0x80000000u;
        d[j] = make_float2(__uint_as_float(__float_as_uint(z.x) ^ s), __uint_as_float(__float_as_uint(z.y) ^ s));
    }
    return outer_bfly<Q>(P, d, m, q);
}

// Q == 1 BPSK: the two samples t0, t1 of a packed pair at once -> xr = (re0, re1), xi = (im0, im1)
template <int DT, int BIT0, int BIT1, bool STAGED>
__device__ __forceinline__ void load_pair_bpsk(const VSrc &src, uint32_t cw, int t0, int t1, float2 &xr, float2 &xi) {
    const uint32_t m0 = bit_mask<BIT0>(cw), m1 = bit_mask<BIT1>(cw);
    if constexpr (DT == DT_SC16) {
        uint32_t w0, w1;
        if constexpr (STAGED) {
            w0 = reinterpret_cast<const uint32_t *>(src.stage)[src.sbase + t0];
            w1 = reinterpret_cast<const uint32_t *>(src.stage)[src.sbase + t1];
        } else {
            w0 = __ldg(reinterpret_cast<const uint32_t *>(src.V) + src.voff + t0);
            w1 = __ldg(reinterpret_cast<const uint32_t *>(src.V) + src.voff + t1);
        }
        sc16_pair_to_f32(w0, w1, m0, m1, xr, xi);
    } else {
        const float2 z0 = fetch_voltage<DT, STAGED>(src, t0), z1 = fetch_voltage<DT, STAGED>(src, t1);
        xr = make_float2(flip_sign(__float_as_uint(z0.x), m0), flip_sign(__float_as_uint(z1.x), m1));
        xi = make_float2(flip_sign(__float_as_uint(z0.y), m0), flip_sign(__float_as_uint(z1.y), m1));
    }
}

// codes[n_ipp][L] (L == Q * 1024 * RA) -> bit-packed words in the fused kernel's pass-A thread order:
// Cbits[p][j][ap * 32 + lane], bit (th * 2 + o) <-> t = j Nk + th 1024 + 64 ap + lane + 32 o.
// *not_bpsk is set to this pre-pass's number `epoch` if any sample is not exactly +-1 + 0j (the fused kernel
// then decodes generally); a flag left by an earlier pre-pass never equals it, so nothing has to be cleared.
__global__ void pack_codes_kernel(const float2 *__restrict__ C, uint32_t *__restrict__ Cbits, int *not_bpsk, int epoch,
                                  int L, int Nk, int RA, int Q, long long total_words) {
    pdl_launch_dependents();                       // the fused kernel's prologue may start now
    const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= total_words) return;
    const int lane = (int)(w & 31), ap = (int)((w >> 5) & 15);
    const long long pj = w >> 9;
    const int j = (int)(pj % Q);
    const long long p = pj / Q;
    const float2 *Crow = C + p * L + (long long)j * Nk + 64 * ap + lane;
    uint32_t bits = 0;
    bool ok = true;
    for (int th = 0; th < RA; th++)
        for (int o = 0; o < 2; o++) {
            const float2 c = __ldg(Crow + th * 1024 + 32 * o);
            ok = ok && (c.y == 0.f) && (c.x == 1.f || c.x == -1.f);
            bits |= (c.x < 0.f ? 1u : 0u) << (th * 2 + o);
        }
    Cbits[w] = bits;
    if (!ok) *not_bpsk = epoch;
}

// ------------------------------------------------------------------------------------------
// N > 16384 (outer radix Q = 2, 4), split path, step 1: decode every window ONCE and apply the outer
// decimation-in-frequency butterfly for all Q residues at once,
//     X[((p R + r) Q + q) Nk + m] = (sum_j d_{p,r}[m + j Nk] W_Q^{jq}) W_N^{mq},   d = V conj(C),
// so that step 2 (the fused kernel on R Q "virtual gates" of length Nk, identity code) reads each decoded
// sample once instead of every (gate, q) CTA decoding the whole window again.
// Outer radix-Q butterfly + twiddles of the two adjacent inner indices m, m + 1 (m even): d[j][k] = decoded sample
// m + k + j Nk; tw[q - 1][k] = W_N^{(m + k) q}.  One 16-byte store per residue at out[q * Nk / 2] (out = the float4
// that holds x_0[m], x_0[m + 1]).
template <int Q>
__device__ __forceinline__ void predecode_combine(const float2 (&d)[Q][2], const float2 (&tw)[Q - 1][2], int Nk, float4 *out) {
    const long long qs = Nk / 2;                                     // float4 elements between residues
    float2 x[Q][2];
#pragma unroll
    for (int k = 0; k < 2; k++) {
        if constexpr (Q == 2) {
            x[0][k] = cadd(d[0][k], d[1][k]);
            x[1][k] = cmul(csub(d[0][k], d[1][k]), tw[0][k]);
        } else {
            static_assert(Q == 4, "outer radix must be 2 or 4");
            const float2 e0 = cadd(d[0][k], d[2][k]), e1 = csub(d[0][k], d[2][k]);
            const float2 o0 = cadd(d[1][k], d[3][k]), o1 = csub(d[1][k], d[3][k]);
            x[0][k] = cadd(e0, o0);
            x[1][k] = cmul(make_float2(e1.x + o1.y, e1.y - o1.x), tw[0][k]);        // e1 - i o1
            x[2][k] = cmul(csub(e0, o0), tw[1][k]);
            x[3][k] = cmul(make_float2(e1.x - o1.y, e1.y + o1.x), tw[2][k]);        // e1 + i o1
        }
    }
#pragma unroll
    for (int q = 0; q < Q; q++) out[q * qs] = make_float4(x[q][0].x, x[q][0].y, x[q][1].x, x[q][1].y);
}

// W_N^{(m + k) q}, q = 1 .. Q - 1, k = 0, 1, from the full-circle table
template <int Q>
__device__ __forceinline__ void predecode_twiddles(const float2 *__restrict__ twN, int m, float2 (&tw)[Q - 1][2]) {
#pragma unroll
    for (int q = 1; q < Q; q++)
#pragma unroll
        for (int k = 0; k < 2; k++) tw[q - 1][k] = __ldg(twN + q * (m + k));
}

// predecode_pair: decode (zero-pad reading A6) + combine for one window; voff = index of the window's
// first sample in V
template <int Q, int DT>
__device__ __forceinline__ void predecode_pair(const void *__restrict__ V, long long voff, const float2 *__restrict__ Crow,
                                               int L, int Nk, const float2 *__restrict__ twN, int m, float4 *out) {
    float2 d[Q][2], tw[Q - 1][2];
#pragma unroll
    for (int j = 0; j < Q; j++)
#pragma unroll
        for (int k = 0; k < 2; k++) {
            const int t = m + k + j * Nk;
            d[j][k] = t < L ? cmul_conj(load_voltage<DT>(V, voff + t), __ldg(Crow + t)) : make_float2(0.f, 0.f);
        }
    predecode_twiddles<Q>(twN, m, tw);
    predecode_combine<Q>(d, tw, Nk, out);
}

// grid = (Nk / 512, ceil(R / GB), IPPs of the batch); a thread takes two adjacent m of GB successive gates: the code
// samples and the outer twiddles of its m are loaded once and stay in registers for all GB windows (they are the
// same for every gate, and with stride << N the gates' echo samples overlap in L1 / L2), so that per decoded sample
// one echo sample is loaded instead of echo + code + twiddles; two gates' loads are in flight at a time.
// Code row of IPP p: P.C + p * P.c_pitch (c_pitch = 0: one code for every IPP, PLSPEC_OPT_SHARED_CODE).
template <int Q, int DT, int GB>
__global__ void __launch_bounds__(256) predecode_kernel(const KParams P, float2 *__restrict__ X) {
    const int m = 2 * (blockIdx.x * 256 + threadIdx.x);
    const int r0g = blockIdx.y * GB;
    const long long p = blockIdx.z;
    const float2 *Crow = P.C + p * P.c_pitch;
    float2 c[Q][2], tw[Q - 1][2];
#pragma unroll
    for (int j = 0; j < Q; j++)
#pragma unroll
        for (int k = 0; k < 2; k++) {
            const int t = m + k + j * P.Nk;
            c[j][k] = t < P.L ? __ldg(Crow + t) : make_float2(0.f, 0.f);
        }
    predecode_twiddles<Q>(P.twN, m, tw);
    const long long vrow = p * P.v_pitch + P.r0;
    const int g_end = (P.R - r0g) < GB ? (P.R - r0g) : GB;
    for (int g = 0; g < g_end; g += 2) {
        const bool two = g + 1 < g_end;
        float2 z[2][Q][2];
#pragma unroll
        for (int u = 0; u < 2; u++) {
            const long long voff = vrow + (long long)(r0g + g + u) * P.stride;
#pragma unroll
            for (int j = 0; j < Q; j++)
#pragma unroll
                for (int k = 0; k < 2; k++) {
                    const int t = m + k + j * P.Nk;
                    z[u][j][k] = (t < P.L && (u == 0 || two)) ? load_voltage<DT>(P.V, voff + t) : make_float2(0.f, 0.f);
                }
        }
#pragma unroll
        for (int u = 0; u < 2; u++) {
            if (u == 1 && !two) break;
            float2 d[Q][2];
#pragma unroll
            for (int j = 0; j < Q; j++)
#pragma unroll
                for (int k = 0; k < 2; k++) d[j][k] = cmul_conj(z[u][j][k], c[j][k]);
            predecode_combine<Q>(d, tw, P.Nk, reinterpret_cast<float4 *>(X + ((p * P.R + r0g + g + u) * Q) * P.Nk + m));
        }
    }
}

// ------------------------------------------------------------------------------------------
// Post-integration products per range gate (SURVEY.md 8(f) NEXT-2; PAPER.md:40-45 Eq. 1, :79 Eq. 8):
// arg max of S over the up-shifted half [k_min, N/2) and the down-shifted half (N/2, N - k_min] (lowest bin
// wins a tie), the mean power S / n_ipp at those bins, and the mean of the remaining bins of
// [k_min, N - k_min] \ {N/2} further than `guard` from either line (float64 sum).  One CTA of 128 threads per gate.
struct ProfileBest { float v; int k; };
__device__ __forceinline__ ProfileBest better(ProfileBest a, ProfileBest b) {
    return (b.v > a.v || (b.v == a.v && b.k < a.k)) ? b : a;
}
constexpr int kProfileThreads = 128;
__global__ void __launch_bounds__(kProfileThreads) profile_kernel(const float *__restrict__ S, int N, int n_ipp, int k_min, int guard,
                                                                  int *__restrict__ k_up, float *__restrict__ p_up,
                                                                  int *__restrict__ k_dn, float *__restrict__ p_dn,
                                                                  float *__restrict__ noise) {
    // One pass over the row in 128-bit loads, software pipelined: the four loads of the next batch are in flight while
    // this batch is searched (against 256 threads x 8 loads and no overlap: 2-10 % faster on the bench shapes,
    // DESIGN.md section 7): both arg maxima and the float64 sum of every searched bin; the few bins within `guard` of
    // the lines are then taken out of the sum again (they are still in L1/L2), so the row crosses HBM once.
    constexpr int T = kProfileThreads, W = T / 32, U = 4;
    __shared__ ProfileBest sb[2][W];
    __shared__ double ssum[W];
    __shared__ int scnt[W];
    __shared__ int sk[2];
    __shared__ double stotal;
    const float *row = S + (long long)blockIdx.x * N;
    const float4 *row4 = reinterpret_cast<const float4 *>(row);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lo = k_min, hi = N - k_min, mid = N / 2, nv = N / 4;
    const ProfileBest none = {-1.f, 0x7fffffff};                       // S >= 0: any bin beats the start value
    ProfileBest up = none, dn = none;
    double acc = 0.0;
    auto take = [&](float v, int f) {
        if (f >= lo && f <= hi && f != mid) {
            const ProfileBest c = {v, f};
            if (f < mid) up = better(up, c); else dn = better(dn, c);
            acc += (double)v;
        }
    };
    auto load = [&](int i) { return i < nv ? __ldg(row4 + i) : make_float4(0.f, 0.f, 0.f, 0.f); };
    float4 v[U], nx[U];
#pragma unroll
    for (int u = 0; u < U; u++) v[u] = load(tid + u * T);
    for (int i0 = tid; i0 < nv; i0 += U * T) {
#pragma unroll
        for (int u = 0; u < U; u++) nx[u] = load(i0 + (U + u) * T);
        // interior vectors: the four bins summed in float32, the four vectors of a batch too (16 bins: at most five
        // roundings of 2^-24 relative on any path, against the 1e-6 the noise floor is good to), everything above in
        // float64
        float fs = 0.f;
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int i = i0 + u * T;
            if (i >= nv) continue;
            const int f0 = 4 * i;
            if (f0 >= lo && f0 + 3 <= hi && (f0 + 3 < mid || f0 > mid)) {   // interior vector: one candidate, one add
                ProfileBest c = {v[u].x, f0};                            // strict >: the lowest bin wins a tie
                if (v[u].y > c.v) c = {v[u].y, f0 + 1};
                if (v[u].z > c.v) c = {v[u].z, f0 + 2};
                if (v[u].w > c.v) c = {v[u].w, f0 + 3};
                if (f0 < mid) up = better(up, c); else dn = better(dn, c);
                fs += (v[u].x + v[u].y) + (v[u].z + v[u].w);
            } else {
                take(v[u].x, f0); take(v[u].y, f0 + 1); take(v[u].z, f0 + 2); take(v[u].w, f0 + 3);
            }
        }
        acc += (double)fs;
#pragma unroll
        for (int u = 0; u < U; u++) v[u] = nx[u];
    }
    auto warp_best = [&]() {
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            ProfileBest u = {__shfl_xor_sync(0xffffffffu, up.v, o), __shfl_xor_sync(0xffffffffu, up.k, o)};
            ProfileBest d = {__shfl_xor_sync(0xffffffffu, dn.v, o), __shfl_xor_sync(0xffffffffu, dn.k, o)};
            up = better(up, u); dn = better(dn, d);
            acc += __shfl_xor_sync(0xffffffffu, acc, o);
        }
    };
    warp_best();
    if (lane == 0) { sb[0][warp] = up; sb[1][warp] = dn; ssum[warp] = acc; }
    __syncthreads();
    // the bins within `guard` of either line (each once, inside the searched range): at most 2 (2 guard + 1)
    const int g = guard < N ? guard : N, wlen = 2 * g + 1;
    const bool one_warp = 2 * wlen <= 32;                               // the usual case: warp 0 finishes the row alone
    if (warp == 0) {
        up = lane < W ? sb[0][lane] : none; dn = lane < W ? sb[1][lane] : none;
        acc = lane < W ? ssum[lane] : 0.0;
        warp_best();                                                    // every lane of warp 0 now holds the row's results
        if (lane == 0) {
            k_up[blockIdx.x] = up.k; k_dn[blockIdx.x] = dn.k;
            p_up[blockIdx.x] = up.v / (float)n_ipp;
            p_dn[blockIdx.x] = dn.v / (float)n_ipp;
            if (!one_warp) { sk[0] = up.k; sk[1] = dn.k; stotal = acc; }
        }
    } else if (one_warp) {
        return;
    }
    if (!one_warp) __syncthreads();
    const int ku = one_warp ? up.k : sk[0], kd = one_warp ? dn.k : sk[1];
    double ex = 0.0;
    int nex = 0;
    for (int j = one_warp ? lane : tid; j < 2 * wlen; j += one_warp ? 32 : T) {
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
    if (!one_warp) {
        if (lane == 0) { ssum[warp] = ex; scnt[warp] = nex; }
        __syncthreads();
        if (tid != 0) return;
        for (int w = 1; w < W; w++) { ex += ssum[w]; nex += scnt[w]; }
        acc = stotal;
    }
    if (tid == 0) {
        const int cnt = (hi - lo) - nex;                               // hi - lo + 1 searched bins less N/2
        noise[blockIdx.x] = cnt > 0 ? (float)((acc - ex) / (double)cnt / (double)n_ipp) : 0.f;
    }
}

// Mean spectrum (Eq. 8, the AVERAGE power), optionally with the zero
// frequency moved to the centre of each row: P[r][g] = S[r][f] / n_ipp, g = f (natural order) or
// g = (f + N/2) mod N (centred).  One read and one write of R N floats, 128-bit and contiguous on both sides
// (N/2 is a multiple of 4): HBM-bound, 8 B per bin.  IEEE division, so that x / 1 = x and both sides of the
// parity test round alike.
__global__ void __launch_bounds__(256) mean_spectrum_kernel(const float4 *__restrict__ S, float4 *__restrict__ P,
                                                            long long n_vec, int log2N, int n_ipp, int centred) {
    const float d = (float)n_ipp;
    const int nv_row = 1 << (log2N - 2), half = centred ? nv_row >> 1 : 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += (long long)gridDim.x * blockDim.x) {
        float4 v = __ldcs(S + i);
        v.x = __fdiv_rn(v.x, d); v.y = __fdiv_rn(v.y, d); v.z = __fdiv_rn(v.z, d); v.w = __fdiv_rn(v.w, d);
        const long long row = i >> (log2N - 2);
        const int c = (int)(i & (nv_row - 1));
        __stcs(P + (row << (log2N - 2)) + ((c + half) & (nv_row - 1)), v);
    }
}

// ------------------------------------------------------------------------------------------
// Diagnostic (SURVEY.md section 7 step 6, 8(d) "measured FMA peak to be reported beside it"): the FP32 FMA issue
// rate of the device, the measured denominator of the ALU roofline.  Every thread runs 32 independent
// multiply-add chains -- 32 scalar FFMA, or 16 packed FFMA2 (the form the fused kernel issues) -- per loop
// iteration: 64 flop per thread and iteration either way.  2048 threads per SM keep every sub-partition's
// FMA pipe full; nothing touches memory inside the loop.
template <bool PACKED>
__global__ void __launch_bounds__(512) fma_peak_kernel(float *__restrict__ out, float a, float b, int iters) {
    float2 acc[16];
#pragma unroll
    for (int j = 0; j < 16; j++) acc[j] = make_float2((float)(threadIdx.x + j), (float)(blockIdx.x - j));
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int j = 0; j < 16; j++) {
            if constexpr (PACKED) {
                acc[j] = __ffma2_rn(acc[j], a2, b2);
            } else {
                acc[j].x = fmaf(acc[j].x, a, b);
                acc[j].y = fmaf(acc[j].y, a, b);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 16; j++) s += acc[j].x + acc[j].y;
    if (s == 1.2345678e-30f) out[0] = s;            // never true for the constants used; keeps the chains alive
}

// Diagnostic: streaming bandwidth with 128-bit accesses (plspec_diag_mem_bandwidth): every CTA of 512 threads walks the
// whole buffer grid-strided, `passes` times.  A buffer below the L2 size measures the SM <-> L2 paths, a large one DRAM.
__global__ void __launch_bounds__(512) bw_read_kernel(const uint4 *__restrict__ a, size_t nvec, int passes, uint4 *sink) {
    uint4 acc = make_uint4(0, 0, 0, 0);
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; p++) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < nvec; i += 4 * stride) {                // four loads in flight per thread, L2 only (no L1)
            const uint4 v0 = __ldcg(a + i), v1 = __ldcg(a + i + stride), v2 = __ldcg(a + i + 2 * stride), v3 = __ldcg(a + i + 3 * stride);
            acc.x ^= v0.x ^ v1.x ^ v2.x ^ v3.x; acc.y ^= v0.y ^ v1.y ^ v2.y ^ v3.y;
            acc.z ^= v0.z ^ v1.z ^ v2.z ^ v3.z; acc.w ^= v0.w ^ v1.w ^ v2.w ^ v3.w;
        }
        for (; i < nvec; i += stride) { const uint4 v = __ldcg(a + i); acc.x ^= v.x; acc.y ^= v.y; acc.z ^= v.z; acc.w ^= v.w; }
    }
    if (acc.x == 0x12345678u && acc.y == 0x9abcdef0u) sink[0] = acc;   // never true for the zero-filled buffer
}
__global__ void __launch_bounds__(512) bw_write_kernel(uint4 *__restrict__ a, size_t nvec, int passes) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; p++) {
        const uint4 v = make_uint4(p, threadIdx.x, blockIdx.x, 7);
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) a[i] = v;
    }
}
// first half of the buffer -> second half
__global__ void __launch_bounds__(512) bw_copy_kernel(uint4 *__restrict__ a, size_t nvec, int passes) {
    const size_t half = nvec / 2, stride = (size_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; p++) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < half; i += 4 * stride) {
            const uint4 v0 = __ldcg(a + i), v1 = __ldcg(a + i + stride), v2 = __ldcg(a + i + 2 * stride), v3 = __ldcg(a + i + 3 * stride);
            a[half + i] = v0; a[half + i + stride] = v1; a[half + i + 2 * stride] = v2; a[half + i + 3 * stride] = v3;
        }
        for (; i < half; i += stride) a[half + i] = __ldcg(a + i);
    }
}
// writes by the TMA engine: thread 0 of every CTA streams its contiguous share of the buffer out of a 2 x 16 KB
// shared-memory staging area with cp.async.bulk stores, four in flight
__global__ void __launch_bounds__(512) bw_tma_store_kernel(unsigned char *__restrict__ a, size_t bytes, int passes) {
    constexpr uint32_t CHUNK = 16384;
    __shared__ __align__(128) unsigned char sm[2 * CHUNK];
    for (int i = threadIdx.x; i < (int)(2 * CHUNK / 4); i += 512) reinterpret_cast<uint32_t *>(sm)[i] = i;
    __syncthreads();
    fence_proxy_async();
    if (threadIdx.x != 0) return;
    const size_t per_cta = (bytes / gridDim.x) & ~(size_t)(CHUNK - 1);
    unsigned char *base = a + (size_t)blockIdx.x * per_cta;
    int k = 0;
    for (int p = 0; p < passes; p++)
        for (size_t off = 0; off < per_cta; off += CHUNK, k++) {
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(base + off),
                         "r"(smem_u32(sm + (k & 1) * CHUNK)), "r"(CHUNK) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 3;" ::: "memory");
        }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
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

}  // namespace plspec
