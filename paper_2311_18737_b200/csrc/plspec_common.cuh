// plspec_common.cuh -- shared device helpers for the plspec kernels (sm_100a).
//
// Notation follows include/plspec.h and the paper: V = received voltages, C = transmit
// code, d = decoded window, X = its length-N DFT,
// S[r][f] = accumulated |X|^2 (Eq. 8).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace plspec {

enum { DT_CF32 = 0, DT_SC16 = 1 };

// Kernel arguments (one struct, passed by value).
struct KParams {
    const void   *V;        // voltages[n_ipp][v_pitch] (float2 or short2 per sample)
    const float2 *C;        // codes[n_ipp][L]
    float        *S;        // S_dev[R][Q][Nk]  (Q = N / Nk outer radix; natural order when Q == 1)
    const float2 *twA;      // fused kernel, pass A -> B1: [a'][f_hi][re/im][lane] pairs W_Nk^{t_lo f_hi}
    const float2 *twB;      // fused kernel, pass B1 -> B2: [c'][re/im][lane] pairs W_1024^{b c}
    const float2 *twN;      // [N]: exp(-2 pi i e / N), full circle
    const uint32_t *Cbits;  // fused kernel, BPSK fast path: [n_ipp][Q][512] packed code signs (or null)
    const int    *not_bpsk; // device flag written by pack_codes_kernel: != epoch -> use Cbits
    int           epoch;    // number of this launch's code pre-pass (never 0; the flag starts at 0)
    long long     v_pitch;  // samples between successive IPP rows of V
    int N, Nk, Q, log2Nk;
    int L;                  // code_len
    int R, r0, stride;
    int n_groups;           // gate groups per launch: ceil(R / gates per CTA)
    int n_ipp, n_chunks;    // IPPs of this launch are split over n_chunks CTAs per (gate, q)
    int use_atomic;         // 1: partial sums meet in S via red.global.add.f32
    // ring mode of the fused kernel (N > 16384, plspec_fused.cuh): the fields above describe the caller's problem
    // (V, C, N, Q = N / Nk, L, R real gates, r0, stride); the decoded residues go through `ring`
    float2 *ring;           // [ring_depth][gridDim.x][Nk] decoded, butterflied windows (stays in L2)
    int    *ring_flags;     // [2][ring_depth] arrival counters, 128 bytes apart: ready, then done
    int ring_depth;         // slots
    int ring_ahead;         // steps a slice is produced ahead of its use
    int c_pitch;            // samples between successive code rows (0: one code for every IPP)
    int ring_stage;         // 1: the producers' inputs go through shared memory (bulk copies one step ahead)
};

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// (a)(b)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * conj(b)  -- the decode multiply of PAPER.md:107 ("takes the conjugate of the transmit
// signal (TX) and complex multiplies that with the corresponding element in the return echo")
__device__ __forceinline__ float2 cmul_conj(float2 a, float2 b) {
    return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// Exact int16 -> fp32 for an interleaved (I, Q) pair packed in one 32-bit word, without the
// quarter-rate I2F pipe: (x ^ 0x8000) is x + 32768 as an unsigned 16-bit value u, and the bit
// pattern 0x4B000000 | u is the float 2^23 + u, so subtracting 2^23 + 32768 gives x exactly.
__device__ __forceinline__ float2 sc16_to_f32(uint32_t w) {
    w ^= 0x80008000u;
    float re = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)) - 8421376.0f;
    float im = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)) - 8421376.0f;
    return make_float2(re, im);
}

// all-ones if bit BIT of w is set, else 0: one shift shared by the four bits at BIT + 8k, then PRMT's
// sign-replicate mode (selector nibble 8 + byte) smears the byte's top bit over the word
template <int BIT>
__device__ __forceinline__ uint32_t bit_mask(uint32_t w) {
    constexpr uint32_t sel = 0x8888u + 0x1111u * (BIT >> 3);
    uint32_t m;
    asm("prmt.b32 %0, %1, 0, %2;" : "=r"(m) : "r"(w << (7 - (BIT & 7))), "n"(sel));   // __byte_perm drops selector bit 3
    return m;
}

// x with its sign bit flipped where the mask (0 or ~0) is set: x ^ (m & 0x80000000) as ONE three-input logic
// operation (left to itself the compiler shares the AND between the two components of a sample: three instructions
// per sample instead of two, on the pipe that limits the decode)
__device__ __forceinline__ float flip_sign(uint32_t x, uint32_t m) {
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, 0x80000000, 0x78;" : "=r"(r) : "r"(x), "r"(m));
    return __uint_as_float(r);
}

// two sc16 samples -> (re0, re1), (im0, im1), negated where the mask (0 or ~0) is set.  -x = ~x + 1 in
// two's complement: complementing both halves of the word gives -x - 1, and the + 1 moves into the constant
// of the packed subtraction (2^23 + 32768 or one less: adjacent fp32 bit patterns).
__device__ __forceinline__ void sc16_pair_to_f32(uint32_t w0, uint32_t w1, uint32_t m0, uint32_t m1, float2 &re,
                                                 float2 &im) {
    w0 ^= 0x80008000u ^ m0;
    w1 ^= 0x80008000u ^ m1;
    const float2 fr = make_float2(__uint_as_float(__byte_perm(w0, 0x4B000000u, 0x7610)),
                                  __uint_as_float(__byte_perm(w1, 0x4B000000u, 0x7610)));
    const float2 fi = make_float2(__uint_as_float(__byte_perm(w0, 0x4B000000u, 0x7632)),
                                  __uint_as_float(__byte_perm(w1, 0x4B000000u, 0x7632)));
    const float2 k = make_float2(__uint_as_float(0xCB008000u + m0), __uint_as_float(0xCB008000u + m1));   // -(2^23 + 32768) [+ 1]
    re = __fadd2_rn(fr, k);
    im = __fadd2_rn(fi, k);
}

// The same conversion through the conversion unit (I2F.S16 with a half-word operand; 16 lanes per clock and SM, its
// own pipe) and one packed multiply by +-1: three ALU-pipe instructions per sample fewer than the form above, at two
// I2F per sample.  Used for every other sample pair where the ALU pipe is the bottleneck (early decode, plspec_fused.cuh).
// Exact like the other: the conversion is exact and so is the product with +-1 (a zero sample may come out as -0).
__device__ __forceinline__ void sc16_pair_to_f32_xu(uint32_t w0, uint32_t w1, uint32_t m0, uint32_t m1, float2 &re, float2 &im) {
    float r0, i0, r1, i1;
    asm("{\n.reg .b16 lo, hi;\nmov.b32 {lo, hi}, %2;\ncvt.rn.f32.s16 %0, lo;\ncvt.rn.f32.s16 %1, hi;\n}" : "=f"(r0), "=f"(i0) : "r"(w0));
    asm("{\n.reg .b16 lo, hi;\nmov.b32 {lo, hi}, %2;\ncvt.rn.f32.s16 %0, lo;\ncvt.rn.f32.s16 %1, hi;\n}" : "=f"(r1), "=f"(i1) : "r"(w1));
    const float2 s = make_float2(__uint_as_float((m0 & 0x80000000u) | 0x3F800000u), __uint_as_float((m1 & 0x80000000u) | 0x3F800000u));
    re = __fmul2_rn(make_float2(r0, r1), s);
    im = __fmul2_rn(make_float2(i0, i1), s);
}

template <int DT>
__device__ __forceinline__ float2 load_voltage(const void *V, long long idx) {
    if constexpr (DT == DT_CF32) {
        return __ldg(reinterpret_cast<const float2 *>(V) + idx);
    } else {
        return sc16_to_f32(__ldg(reinterpret_cast<const uint32_t *>(V) + idx));
    }
}

// ---- mbarrier + bulk async copy (TMA, 1-D): global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// generic-proxy accesses before this fence are ordered before later async-proxy (bulk copy) accesses
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t mbar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t mbar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(mbar), "r"(parity) : "memory");
}
// dst, src 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(mbar)
                 : "memory");
}

// ---- tensor memory (TMEM) used as a per-thread constant store: 128 lanes x 512 columns x 32 bit per SM.
// A warp reaches the 32 lanes of quadrant (warp % 4); `32x32b` gives thread i lane (quadrant base + i),
// consecutive columns.  Address = (lane << 16) | column.
__device__ __forceinline__ void tmem_alloc_512(uint32_t smem_result_addr) {          // one whole warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_result_addr) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_512(uint32_t taddr) {                     // one whole warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_st4(uint32_t a, float x0, float x1, float x2, float x3) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(x0), "f"(x1), "f"(x2), "f"(x3) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// 8 consecutive columns -> v[0..7]; the values may be used only after tmem_wait_ld8(v)
__device__ __forceinline__ void tmem_ld8(uint32_t a, float (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "r"(a));
}
__device__ __forceinline__ void tmem_wait_ld8(float (&v)[8]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(v[0]), "+f"(v[1]), "+f"(v[2]), "+f"(v[3]), "+f"(v[4]), "+f"(v[5]), "+f"(v[6]), "+f"(v[7]));
}
// ---- cross-CTA hand-over through global memory (ring mode): release / acquire at gpu scope
__device__ __forceinline__ void red_release_add(int *p, int v) {
    asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_acquire(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// ... and inside the CTA (shared memory, cta scope): arrival counting and a published progress word
__device__ __forceinline__ int atom_add_acq_rel_cta(uint32_t saddr, int v) {
    int old;
    asm volatile("atom.acq_rel.cta.shared::cta.add.s32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ int atom_cas_acquire_cta(uint32_t saddr, int cmp, int v) {
    int old;
    asm volatile("atom.acquire.cta.shared::cta.cas.b32 %0, [%1], %2, %3;" : "=r"(old) : "r"(saddr), "r"(cmp), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ int ld_acquire_cta(uint32_t saddr) {
    int v;
    asm volatile("ld.acquire.cta.shared::cta.s32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta(uint32_t saddr, int v) {
    asm volatile("st.release.cta.shared::cta.s32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory");
}
// Programmatic dependent launch: a kernel launched with the stream-serialisation attribute may start while
// its predecessor in the stream is still running; it must not touch anything the predecessor (or any earlier
// work) writes before pdl_wait() returns.  Both are no-ops in a plain launch.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// compile-time loop
template <int B, int E, class F>
__device__ __forceinline__ void sfor(F &&f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        sfor<B + 1, E>(f);
    }
}

template <int LOG>
__host__ __device__ constexpr int brev(int j) {
    int r = 0;
    for (int b = 0; b < LOG; b++) r |= ((j >> b) & 1) << (LOG - 1 - b);
    return r;
}
__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }

}  // namespace plspec
