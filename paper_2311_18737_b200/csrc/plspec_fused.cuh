// plspec_fused.cuh -- the fused decode + FFT + |X|^2 + accumulate kernel.
//
// One CTA = 16 warps = 16 warp-local 1024-point FFTs.  Nk = 1024 * RA (RA = 1, 2, 4, 8, 16) is the
// length one CTA transforms per window, so a CTA works on G = 16 / RA range gates at a time; N = Q * Nk
// with an outer radix Q = 1, 2, 4 folded into the load (decimation in frequency, as in the header of
// plspec_kernels.cuh).  The S accumulators of the CTA's gates stay in registers across all IPPs of
// the tile and reach HBM once, at the end (PAPER.md:115 accumulates per pulse in device memory).
//
// Index algebra (forward DFT, W_n = exp(-2 pi i / n); d = decoded window):
//   inner index m = t_hi * 1024 + t_lo,  t_lo = 32 a + b,   output k = f_hi + RA * (c + 32 e)
//   pass A  (thread <-> two t_lo 32 apart, all t_hi):
//       y_{f_hi}[t_lo] = W_Nk^{t_lo f_hi} * sum_{t_hi} x[t_hi * 1024 + t_lo] W_RA^{t_hi f_hi}
//   pass B1 (warp <-> (gate, f_hi), lane = b):  z[c][b] = W_1024^{b c} * sum_a y[32 a + b] W_32^{a c}
//   pass B2 (same warp, lane = c):              X[f_hi + RA (c + 32 e)] = sum_b z[c][b] W_32^{b e}
//
// Arithmetic is packed: every float2 holds the SAME component (re or im) of TWO complex values
// that go through identical butterflies (FADD2 / FMUL2 / FFMA2 on sm_100a: two lane-operations per
// issue slot).  Pairs: pass A -- the thread's two t_lo (a even / a odd); B1 -- the even-a and odd-a
// halves of a decimation-in-time radix-32; B2 -- the sum and difference halves of a
// decimation-in-frequency radix-32, which are the even and odd output bins e.
// Butterflies with a non-trivial constant twiddle use the 6-FMA form
//   a +- W b = a +- wc * (b_r + t b_i,  b_i - t b_r),  t = tan,   (or the cotangent form when |ws| > |wc|)
// with wc and t as FFMA2 immediates.
//
// Shared memory: 16 regions (one per B warp) of 16*65 8-byte slots + the B1->B2 twiddle table.
//   A -> B1 :  slot (a'*2 + plane)*32 + b        holds (y[32(2a')+b], y[32(2a'+1)+b]).plane      (STS.64 / LDS.64)
//              RA >= 4: 16-byte slot a'*32 + b   holds both planes of that pair                    (STS.128 / LDS.128)
//   B1 -> B2:  slot  bb*65 + plane*32 + c        holds (z[c][bb], z[c][bb+16]).plane             (STS.32 / LDS.64)
// Both are free of bank conflicts (the 65 pitch spreads the 4-byte transposed stores over all banks).
//
// S_dev layout written by this kernel: [r][q][f_hi][e][c]  (c = lane: every flush is 128 B per warp);
// finalize_kernel restores natural bin order at finalize.
#pragma once
#include "plspec_common.cuh"

namespace plspec {

// A -> B1: 16 x 32 slots of 16 bytes (8192); B1 -> B2: 16 x 65 slots of 8 bytes (8320), or, where pass B2 is the
// decimation-in-time form (B2D in the kernel), 64 rows (plane, c) of 32 words at a pitch of 34 (8704)
constexpr int kRegionBytes = 16 * 65 * 8;                    // 8320
constexpr int kRegionBytesDit = 64 * 34 * 4;                 // 8704: the kernel whose pass B2 is decimation in time
constexpr int kDitExtraBytes = 16 * (kRegionBytesDit - kRegionBytes);   // what that kernel needs beyond kStageOff
constexpr int kFusedSmemBytes = 16 * kRegionBytes;
// control words: stage mbarrier (8) + warp arrival counter (4) + TMEM base (4) + per region a "free" and a
// "full" mbarrier
// + ring mode: per-CTA arrival counters (ready x 4, done x 4), progress words (ready, free) and their poller locks
constexpr int kRingCtlOff = 16 + 32 * 8;
constexpr int kStageCtlBytes = kRingCtlOff + 64;
constexpr int kStageOff = kFusedSmemBytes + kStageCtlBytes;    // voltage stage of the ST variant (16-byte aligned)
constexpr int kSmemMax = 227 * 1024;
constexpr int kStageMaxBytes = kSmemMax - kStageOff;
constexpr int kFusedThreads = 512;
constexpr int kRingFlushEvery = 10;

// ---- compile-time cos / sin of 2 pi k / 32 (float64, correctly rounded literals)
constexpr double kCos32d[9] = {1.0,
                               0.98078528040323044913,
                               0.92387953251128675613,
                               0.83146961230254523708,
                               0.70710678118654752440,
                               0.55557023301960222474,
                               0.38268343236508977173,
                               0.19509032201612826785,
                               0.0};
__host__ __device__ constexpr double cosd32(int k) {
    k = ((k % 32) + 32) % 32;
    if (k > 16) k = 32 - k;
    return k > 8 ? -kCos32d[16 - k] : kCos32d[k];
}
__host__ __device__ constexpr double sind32(int k) { return cosd32(k - 8); }
__host__ __device__ constexpr double absd(double x) { return x < 0 ? -x : x; }

// ---- packed helpers: a float2 is two independent lanes
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 pmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 pfmak(float2 a, float k, float2 c) { return __ffma2_rn(a, make_float2(k, k), c); }
__device__ __forceinline__ float2 pneg(float2 a) { return make_float2(-a.x, -a.y); }

// (a, b) -> (a + W b, a - W b),  W = W_32^K32 = cos - i sin,  on two packed complex values at once
template <int K32>
__device__ __forceinline__ void bfly_dit(float2 &ar, float2 &ai, float2 &br, float2 &bi) {
    if constexpr (K32 == 0) {
        const float2 tr = br, ti = bi;
        br = psub(ar, tr); bi = psub(ai, ti);
        ar = padd(ar, tr); ai = padd(ai, ti);
    } else if constexpr (K32 == 8) {                       // W = -i:  W b = (b_i, -b_r)
        const float2 tr = bi, ti = br;
        br = psub(ar, tr); bi = padd(ai, ti);
        ar = padd(ar, tr); ai = psub(ai, ti);
    } else {
        constexpr double c = cosd32(K32), s = sind32(K32);
        if constexpr (absd(c) >= absd(s)) {
            constexpr float t = (float)(s / c), w = (float)c;   // W b = w (b_r + t b_i, b_i - t b_r)
            const float2 p = pfmak(bi, t, br), q = pfmak(br, -t, bi);
            br = pfmak(p, -w, ar); bi = pfmak(q, -w, ai);
            ar = pfmak(p, w, ar);  ai = pfmak(q, w, ai);
        } else {
            constexpr float t = (float)(c / s), w = (float)s;   // W b = w (t b_r + b_i, t b_i - b_r)
            const float2 p = pfmak(br, t, bi), q = pfmak(bi, t, pneg(br));
            br = pfmak(p, -w, ar); bi = pfmak(q, -w, ai);
            ar = pfmak(p, w, ar);  ai = pfmak(q, w, ai);
        }
    }
}

// Radix-2 decimation-in-time DFT of n = 1..16 packed points held at r[OFF..OFF+n), i[OFF..OFF+n) in
// natural order; on return X[k] sits at index OFF + brev(k).
template <int n, int OFF, int M>
__device__ __forceinline__ void dft_packed(float2 (&r)[M], float2 (&i)[M]) {
    constexpr int LOG = ilog2(n);
    sfor<0, LOG>([&](auto s_) {
        constexpr int half = 1 << decltype(s_)::value, len = 2 * half;
        sfor<0, n / 2>([&](auto t_) {
            constexpr int t = decltype(t_)::value;
            constexpr int k = t % half, base = (t / half) * len;
            constexpr int ia = OFF + brev<LOG>(base + k), ib = OFF + brev<LOG>(base + k + half);
            bfly_dit<k * (32 / len)>(r[ia], i[ia], r[ib], i[ib]);
        });
    });
}

// Last stage of the packed 16-point DIT fused with |X|^2 (Eq. 8): the butterfly outputs a +- W b
// are never formed.  |a +- W b|^2 = (|a|^2 + |b|^2) +- 2 Re(conj(a) W b), so per butterfly two running sums
//   accS += |a|^2 + |b|^2,   accC += a_r p + a_i q   with  W b = w (p, q)  (tangent / cotangent form)
// replace four adds and four multiply-adds by six multiply-adds (eight with a non-trivial twiddle instead of
// ten); the two spectra values are accS +- 2 w accC at flush time (kPow2w).
template <int K32>
__device__ __forceinline__ void bfly_power(float2 ar, float2 ai, float2 br, float2 bi, float2 &accS, float2 &accC) {
    accS = pfma(ar, ar, accS); accS = pfma(ai, ai, accS);
    accS = pfma(br, br, accS); accS = pfma(bi, bi, accS);
    if constexpr (K32 == 0) {
        accC = pfma(ar, br, accC); accC = pfma(ai, bi, accC);
    } else if constexpr (K32 == 8) {                       // W b = (b_i, -b_r)
        accC = pfma(ar, bi, accC); accC = pfma(ai, pneg(br), accC);
    } else {
        constexpr double c = cosd32(K32), sn = sind32(K32);
        if constexpr (absd(c) >= absd(sn)) {
            constexpr float t = (float)(sn / c);
            const float2 p = pfmak(bi, t, br), q = pfmak(br, -t, bi);
            accC = pfma(ar, p, accC); accC = pfma(ai, q, accC);
        } else {
            constexpr float t = (float)(c / sn);
            const float2 p = pfmak(br, t, bi), q = pfmak(bi, t, pneg(br));
            accC = pfma(ar, p, accC); accC = pfma(ai, q, accC);
        }
    }
}
// 2 w of the butterfly above: w = 1 for the trivial twiddles, else cos or sin (whichever is larger in modulus)
__host__ __device__ constexpr float pow2w(int K32) {
    if (K32 == 0 || K32 == 8) return 2.0f;
    const double c = cosd32(K32), sn = sind32(K32);
    return (float)(2.0 * (absd(c) >= absd(sn) ? c : sn));
}

// Last stage of a decimation-in-time radix-32 whose halves sit in one register pair, (.x, .y) = (E, O), fused with
// |X|^2: X[e] = E + W O, X[e + 16] = E - W O, W = W_32^K32, so |X|^2 = (|E|^2 + |O|^2) +- 2 Re(conj(E) W O) with
// W O = w (p, q) in the tangent / cotangent form: accS += |E|^2 + |O|^2, accC += E_r p + E_i q; the two spectra values
// are accS +- 2 w accC at flush time (pow2w).
template <int K32>
__device__ __forceinline__ void bfly_power_halves(float2 r, float2 i, float &accS, float &accC) {
    const float er = r.x, ei = i.x, orr = r.y, oi = i.y;
    accS = fmaf(er, er, accS); accS = fmaf(ei, ei, accS);
    accS = fmaf(orr, orr, accS); accS = fmaf(oi, oi, accS);
    if constexpr (K32 == 0) {
        accC = fmaf(er, orr, accC); accC = fmaf(ei, oi, accC);
    } else if constexpr (K32 == 8) {                       // W O = (O_i, -O_r)
        accC = fmaf(er, oi, accC); accC = fmaf(-ei, orr, accC);
    } else {
        constexpr double c = cosd32(K32), sn = sind32(K32);
        float p, q;
        if constexpr (absd(c) >= absd(sn)) {
            constexpr float t = (float)(sn / c);
            p = fmaf(oi, t, orr); q = fmaf(orr, -t, oi);
        } else {
            constexpr float t = (float)(c / sn);
            p = fmaf(orr, t, oi); q = fmaf(oi, t, -orr);
        }
        accC = fmaf(er, p, accC); accC = fmaf(ei, q, accC);
    }
}

// the first LOG - 1 stages of dft_packed<16, 0>
template <int M>
__device__ __forceinline__ void dft_packed16_head(float2 (&r)[M], float2 (&i)[M]) {
    sfor<0, 3>([&](auto s_) {
        constexpr int half = 1 << decltype(s_)::value, len = 2 * half;
        sfor<0, 8>([&](auto t_) {
            constexpr int t = decltype(t_)::value;
            constexpr int k = t % half, base = (t / half) * len;
            constexpr int ia = brev<4>(base + k), ib = brev<4>(base + k + half);
            bfly_dit<k * (32 / len)>(r[ia], i[ia], r[ib], i[ib]);
        });
    });
}

// last stage of a decimation-in-time radix-32: (.x, .y) = (E, O) -> (E + W O, E - W O), W = W_32^K32
template <int K32>
__device__ __forceinline__ void bfly_dit_halves(float2 &r, float2 &i) {
    const float er = r.x, ei = i.x, orr = r.y, oi = i.y;
    if constexpr (K32 == 0) {
        r.x = er + orr; r.y = er - orr; i.x = ei + oi; i.y = ei - oi;
    } else if constexpr (K32 == 8) {
        r.x = er + oi; r.y = er - oi; i.x = ei - orr; i.y = ei + orr;
    } else {
        constexpr double c = cosd32(K32), s = sind32(K32);
        float p, q, w;
        if constexpr (absd(c) >= absd(s)) {
            constexpr float t = (float)(s / c);
            w = (float)c; p = fmaf(oi, t, orr); q = fmaf(orr, -t, oi);
        } else {
            constexpr float t = (float)(c / s);
            w = (float)s; p = fmaf(orr, t, oi); q = fmaf(oi, t, -orr);
        }
        r.x = fmaf(p, w, er); r.y = fmaf(p, -w, er);
        i.x = fmaf(q, w, ei); i.y = fmaf(q, -w, ei);
    }
}

// first stage of a decimation-in-frequency radix-32: (.x, .y) = (z0, z1) -> (z0 + z1, (z0 - z1) W_32^K32)
template <int K32>
__device__ __forceinline__ void bfly_dif_halves(float2 &r, float2 &i) {
    const float ur = r.x + r.y, ui = i.x + i.y, dr = r.x - r.y, di = i.x - i.y;
    r.x = ur; i.x = ui;
    if constexpr (K32 == 0) {
        r.y = dr; i.y = di;
    } else if constexpr (K32 == 8) {
        r.y = di; i.y = -dr;
    } else {
        constexpr float c = (float)cosd32(K32), s = (float)sind32(K32);
        r.y = fmaf(s, di, c * dr);
        i.y = fmaf(-s, dr, c * di);
    }
}

// ------------------------------------------------------------------------------------------
// Ring mode (fused_kernel with RQ = 2, 4; see there), producer side.  These are real functions (not inlined): their
// working set must not compete with the register allocation of the transform loop that calls them.
//
// Producer inputs through shared memory (P.ring_stage != 0: they fit): the code samples and the run of echo samples
// this CTA's slice needs for step sp are brought in by bulk asynchronous copies (TMA) two steps ahead, into buffer
// sp & 1, so that the decode reads shared memory instead of waiting on L2; its outer twiddles, which never change
// (the slice of m is fixed), are loaded once.  Layout per buffer: RQ code rows of `cp` float2, then RQ echo rows of
// `vb` bytes; every row starts at the 16-byte boundary at or below its first element (as in the ST variant).
template <int RQ, int VDT>
struct RingGeo {
    static constexpr int NK = 16384, VESZ = VDT == DT_CF32 ? 8 : 4;
    int mp0, npair, npmax, GR, cp, vb, buf;
    unsigned char *stage;
    float2 *tws;                                   // [RQ - 1][2 npmax]
    uint32_t ctl;                                  // ring control words (shared-memory address)
    __device__ __forceinline__ RingGeo(const KParams *P, unsigned char *smem) {
        mp0 = (int)(((long long)blockIdx.x * (NK / 2)) / gridDim.x);
        npair = (int)((((long long)blockIdx.x + 1) * (NK / 2)) / gridDim.x) - mp0;
        npmax = (NK / 2 + (int)gridDim.x - 1) / (int)gridDim.x;
        GR = (int)gridDim.x / RQ;
        cp = 2 * npmax + 2;
        vb = (((GR - 1) * P->stride + 2 * npmax) * VESZ + 31) & ~15;
        buf = RQ * (cp * 8 + vb);
        stage = smem + kStageOff;
        tws = reinterpret_cast<float2 *>(stage + 2 * buf);
        ctl = smem_u32(smem + kFusedSmemBytes + kRingCtlOff);
    }
};

// one thread: the bulk copies of step sp into buffer sp & 1, counted on that buffer's mbarrier
template <int RQ, int VDT>
__device__ __noinline__ void ring_stage_issue_fn(const KParams *P, int sp) {
    extern __shared__ __align__(16) unsigned char smem[];
    const RingGeo<RQ, VDT> G(P, smem);
    constexpr int VESZ = RingGeo<RQ, VDT>::VESZ, NK = RingGeo<RQ, VDT>::NK;
    const uint32_t mb = G.ctl + 48 + 8 * (uint32_t)(sp & 1);
    const int kk = sp / P->n_ipp, pp = sp - kk * P->n_ipp;
    const int g_first = kk * G.GR;
    const int gr = (P->R - g_first) < G.GR ? (P->R - g_first) : G.GR;
    const unsigned char *cs[RQ], *vs[RQ];
    uint32_t cb[RQ], vbytes[RQ], total = 0;
#pragma unroll
    for (int j = 0; j < RQ; j++) {
        const int t0 = 2 * G.mp0 + j * NK;
        int valid = P->L - t0;
        valid = valid < 0 ? 0 : (valid > 2 * G.npair ? 2 * G.npair : valid);
        const unsigned char *c = reinterpret_cast<const unsigned char *>(P->C + (long long)pp * P->c_pitch + t0);
        const unsigned char *v = reinterpret_cast<const unsigned char *>(P->V) +
                                 ((long long)pp * P->v_pitch + P->r0 + (long long)g_first * P->stride + t0) * VESZ;
        const uint32_t cm = (uint32_t)(reinterpret_cast<uintptr_t>(c) & 15), vm = (uint32_t)(reinterpret_cast<uintptr_t>(v) & 15);
        cs[j] = c - cm; vs[j] = v - vm;
        cb[j] = valid ? ((cm + (uint32_t)valid * 8 + 15u) & ~15u) : 0u;
        vbytes[j] = valid ? ((vm + (uint32_t)((gr - 1) * P->stride + valid) * VESZ + 15u) & ~15u) : 0u;
        total += cb[j] + vbytes[j];
    }
    mbar_arrive_expect_tx(mb, total);
    unsigned char *buf = G.stage + (sp & 1) * G.buf;
#pragma unroll
    for (int j = 0; j < RQ; j++) {
        if (cb[j]) bulk_g2s(smem_u32(buf + j * G.cp * 8), cs[j], cb[j], mb);
        if (vbytes[j]) bulk_g2s(smem_u32(buf + RQ * G.cp * 8 + j * G.vb), vs[j], vbytes[j], mb);
    }
}

// whole CTA, once: the slice's outer twiddles W_N^{m q}, and the copies of the first two steps
template <int RQ, int VDT>
__device__ __noinline__ void ring_stage_prologue_fn(const KParams *P, int T) {
    extern __shared__ __align__(16) unsigned char smem[];
    const RingGeo<RQ, VDT> G(P, smem);
    for (int i = threadIdx.x; i < (RQ - 1) * 2 * G.npair; i += kFusedThreads) {
        const int q = i / (2 * G.npair) + 1, mm = i - (q - 1) * 2 * G.npair;
        G.tws[(q - 1) * 2 * G.npmax + mm] = __ldg(P->twN + q * (2 * G.mp0 + mm));
    }
    if (threadIdx.x == 0) {
        fence_proxy_async();
        ring_stage_issue_fn<RQ, VDT>(P, 0);
        if (T > 1) ring_stage_issue_fn<RQ, VDT>(P, 1);
    }
}

// every warp: this CTA's slice of every window of step sp -> ring slot sp % depth (decode, + outer
// radix-RQ butterfly, plspec_kernels.cuh).  thread <-> (pair of inner indices, set of gates): the code samples and
// twiddles of a pair are read once and serve all the thread's gates.  part 0: the thread's first two gates, 1: the
// rest, -1: all.
template <int RQ, int VDT>
__device__ __noinline__ void ring_produce_fn(const KParams *P, int sp, int part) {
    extern __shared__ __align__(16) unsigned char smem[];
    const RingGeo<RQ, VDT> G(P, smem);
    constexpr int VESZ = RingGeo<RQ, VDT>::VESZ, NKc = RingGeo<RQ, VDT>::NK;
    const int tid = threadIdx.x;
    const bool staged = P->ring_stage != 0;
    const int L = P->L, stride = P->stride;
    const int kk = sp / P->n_ipp, pp = sp - kk * P->n_ipp;
    const int g_first = kk * G.GR;
    const int gr = (P->R - g_first) < G.GR ? (P->R - g_first) : G.GR;
    const int npair = G.npair, mp0 = G.mp0;
    const int lanes_m = npair < kFusedThreads ? npair : kFusedThreads;
    const int ngs = kFusedThreads / lanes_m;
    const int my_gs = tid / lanes_m, my_m = tid - my_gs * lanes_m;
    float2 *base = P->ring + (size_t)(sp % P->ring_depth) * gridDim.x * (size_t)NKc;
    const float2 *Crow = P->C + (long long)pp * P->c_pitch;
    const long long vrow = (long long)pp * P->v_pitch + P->r0;
    const unsigned char *sbuf = G.stage + (sp & 1) * G.buf;
    int cmis[RQ], vmis[RQ];
    if (staged) {                                  // wait for this step's copies; element index of sample (m - 2 mp0) in row j = mis_j + ...
        mbar_wait(G.ctl + 48 + 8 * (uint32_t)(sp & 1), (uint32_t)(sp >> 1) & 1u);
#pragma unroll
        for (int j = 0; j < RQ; j++) {
            const int t0 = 2 * mp0 + j * NKc;
            cmis[j] = (int)((reinterpret_cast<uintptr_t>(Crow + t0) & 15) >> 3);
            vmis[j] = (int)((reinterpret_cast<uintptr_t>(reinterpret_cast<const unsigned char *>(P->V) +
                                                        (vrow + (long long)g_first * stride + t0) * VESZ) & 15) / VESZ);
        }
    }
    if (my_gs >= ngs) return;
    for (int mp = my_m; mp < npair; mp += lanes_m) {
        const int m = 2 * (mp0 + mp);
        float2 c[RQ][2], tw[RQ - 1][2];
#pragma unroll
        for (int j = 0; j < RQ; j++)
#pragma unroll
            for (int k = 0; k < 2; k++) {
                const int t = m + k + j * NKc;
                if (staged)
                    c[j][k] = t < L ? reinterpret_cast<const float2 *>(sbuf + j * G.cp * 8)[cmis[j] + 2 * mp + k] : make_float2(0.f, 0.f);
                else
                    c[j][k] = t < L ? __ldg(Crow + t) : make_float2(0.f, 0.f);
            }
        if (staged) {
#pragma unroll
            for (int q = 1; q < RQ; q++)
#pragma unroll
                for (int k = 0; k < 2; k++) tw[q - 1][k] = G.tws[(q - 1) * 2 * G.npmax + 2 * mp + k];
        } else {
            predecode_twiddles<RQ>(P->twN, m, tw);
        }
        const int tt_lo = part == 1 ? my_gs + 2 * ngs : my_gs, tt_hi = part == 0 ? (gr < my_gs + 2 * ngs ? gr : my_gs + 2 * ngs) : gr;
        for (int tt = tt_lo; tt < tt_hi; tt += ngs) {
            const long long voff = vrow + (long long)(g_first + tt) * stride;
            float2 d[RQ][2];
#pragma unroll
            for (int j = 0; j < RQ; j++)
#pragma unroll
                for (int k = 0; k < 2; k++) {
                    const int t = m + k + j * NKc;
                    float2 z;
                    if (staged) {
                        const int e = vmis[j] + tt * stride + 2 * mp + k;
                        const unsigned char *row = sbuf + RQ * G.cp * 8 + j * G.vb;
                        if constexpr (VDT == DT_CF32)
                            z = t < L ? reinterpret_cast<const float2 *>(row)[e] : make_float2(0.f, 0.f);
                        else
                            z = t < L ? sc16_to_f32(reinterpret_cast<const uint32_t *>(row)[e]) : make_float2(0.f, 0.f);
                    } else {
                        z = t < L ? load_voltage<VDT>(P->V, voff + t) : make_float2(0.f, 0.f);
                    }
                    d[j][k] = cmul_conj(z, c[j][k]);
                }
            predecode_combine<RQ>(d, tw, NKc, reinterpret_cast<float4 *>(base + (size_t)(tt * RQ) * NKc + m));
        }
    }
}

// The common case of ring_produce_fn, kept lean: inputs staged in shared memory, code_len == N (no zero padding), and
// at most one pair of inner indices per thread (gridDim.x >= 16).  Same arithmetic, same order.
template <int RQ, int VDT>
__device__ __noinline__ void ring_produce_lean_fn(const KParams *P, int sp, int part) {
    extern __shared__ __align__(16) unsigned char smem[];
    const RingGeo<RQ, VDT> G(P, smem);
    constexpr int VESZ = RingGeo<RQ, VDT>::VESZ, NKc = RingGeo<RQ, VDT>::NK;
    const int tid = threadIdx.x;
    const int n_ipp = P->n_ipp, stride = P->stride;
    const int kk = sp / n_ipp, pp = sp - kk * n_ipp;
    const int g_first = kk * G.GR;
    const int gr = (P->R - g_first) < G.GR ? (P->R - g_first) : G.GR;
    const int npair = G.npair;
    const int ngs = kFusedThreads / npair;
    const int my_gs = tid / npair, mp = tid - my_gs * npair;
    const unsigned char *sbuf = G.stage + (sp & 1) * G.buf;
    mbar_wait(G.ctl + 48 + 8 * (uint32_t)(sp & 1), (uint32_t)(sp >> 1) & 1u);
    if (my_gs >= ngs) return;
    const int tt_lo = part == 1 ? my_gs + 2 * ngs : my_gs, tt_hi = part == 0 ? (gr < my_gs + 2 * ngs ? gr : my_gs + 2 * ngs) : gr;
    if (tt_lo >= tt_hi) return;
    // row j of the buffer starts at the 16-byte boundary at or below its first element: element index = mis_j + ...
    const uintptr_t c0 = reinterpret_cast<uintptr_t>(P->C + (long long)pp * P->c_pitch + 2 * G.mp0);
    const uintptr_t v0 = reinterpret_cast<uintptr_t>(P->V) +
                         (uintptr_t)(((long long)pp * P->v_pitch + P->r0 + (long long)g_first * stride + 2 * G.mp0) * VESZ);
    float2 c[RQ][2], tw[RQ - 1][2];
    const unsigned char *vrow[RQ];
#pragma unroll
    for (int j = 0; j < RQ; j++) {
        // N = RQ * 16384 samples of 8 (4) bytes apart: every row has the misalignment of row 0
        const float2 *cj = reinterpret_cast<const float2 *>(sbuf + j * G.cp * 8) + (int)((c0 & 15) >> 3) + 2 * mp;
        c[j][0] = cj[0];
        c[j][1] = cj[1];
        vrow[j] = sbuf + RQ * G.cp * 8 + j * G.vb + ((int)((v0 & 15) / VESZ) + 2 * mp + tt_lo * stride) * VESZ;
    }
#pragma unroll
    for (int q = 1; q < RQ; q++) {
        tw[q - 1][0] = G.tws[(q - 1) * 2 * G.npmax + 2 * mp];
        tw[q - 1][1] = G.tws[(q - 1) * 2 * G.npmax + 2 * mp + 1];
    }
    float4 *out = reinterpret_cast<float4 *>(P->ring + ((size_t)(sp % P->ring_depth) * gridDim.x + (size_t)(tt_lo * RQ)) * (size_t)NKc +
                                             2 * (G.mp0 + mp));
    const int vstep = ngs * stride * VESZ;
    const size_t ostep = (size_t)ngs * RQ * (NKc / 2);               // float4 elements between successive gates of a thread
    for (int tt = tt_lo; tt < tt_hi; tt += ngs) {
        float2 d[RQ][2];
#pragma unroll
        for (int j = 0; j < RQ; j++) {
#pragma unroll
            for (int k = 0; k < 2; k++) {
                float2 z;
                if constexpr (VDT == DT_CF32) z = reinterpret_cast<const float2 *>(vrow[j])[k];
                else z = sc16_to_f32(reinterpret_cast<const uint32_t *>(vrow[j])[k]);
                d[j][k] = cmul_conj(z, c[j][k]);
            }
            vrow[j] += vstep;
        }
        predecode_combine<RQ>(d, tw, NKc, out);
        out += ostep;
    }
}

// ------------------------------------------------------------------------------------------
// ST = true: the samples of IPP p that the CTA's gates touch (one contiguous run, overlapping windows
// included once) are copied global -> shared by one cp.async.bulk per 32 KB while the CTA is still
// transforming IPP p - 1; pass A then reads shared memory.  The copy starts at the 16-byte boundary at
// or below the first sample and ends at the one at or above the last (CUDA allocations are 256-byte
// granular, so the rounded run never leaves the allocation that holds the samples).
// PFE = false: no prefetch of the next window (below).  The prefetch reads all N samples of a window whatever the
// code length, so the host selects it only when code_len == N (plspec_api.cu: select_kernel): with a shorter code
// (zero-pad reading A6) the last windows of V would be read past the end of the caller's buffer.
//
// RQ = 2, 4: RING MODE for N = RQ * 16384 (RA = 16, Q = 1, DT = CF32, no stage, no prefetch; VDT = the caller's voltage
// dtype).  A CTA can hold the accumulators of only one residue q of a window (X[RQ k + q] = DFT_Nk(x_q)[k],
// plspec_kernels.cuh), yet every residue needs all N decoded samples.  So the grid (cooperative launch, one CTA per SM,
// gridDim.x a multiple of RQ) works in lockstep: in round k CTA c owns the virtual gate vg = k gridDim.x + c
// (gate vg / RQ, residue vg % RQ) for all IPPs; a STEP is one IPP of one round.  For step s every CTA decodes its
// 1 / gridDim.x slice of the inner index m of ALL windows of the round (so the code samples and the overlapping echo
// samples it needs are shared by the round's gates and stay in L1), applies the outer radix-RQ butterfly and writes
// the RQ residues into slot s % depth of a ring in global memory that is small enough to stay in L2; it then
// transforms its own virtual gate's window of step s - ahead.. from the ring like any 16384-point window.  Hand-over:
// per slot a `ready` counter (one release-add per warp after its stores; consumers acquire-poll until all
// 16 gridDim.x warps of the step have arrived) and a `done` counter (one add per warp after its last load of the
// slot; producers wait for it before they overwrite the slot, `depth` steps later).  Counters are monotonic:
// slot i serves steps i, i + depth, ... and step s completes at (s / depth + 1) * 16 gridDim.x.  A CTA never waits for
// a step that needs its own later work, so the grid cannot deadlock as long as all CTAs are resident.
// The decoded windows never reach DRAM: the scratch round trip of the old split path (2 x 21 GB at cfg 4) is gone.
// IDC = true: identity code -- the windows are decoded already (step 2 of the scratch path for N > 16384): pass A
// takes the prefetched complex64 words as they are (no code words, no sign flips).
// ED = true: EARLY DECODE (staged variants, Q = 1; +-1 codes).  The stage puts the next window's raw samples a
// shared-memory load away while the current window is still in pass B2, and the last butterfly stage retires eight
// registers per step.  So the next window is decoded right there: after step k of the last stage the two sample
// pairs whose registers just died are read from the stage, converted and sign-flipped (PRMT / LOP3 / IADD3: the
// half-rate ALU pipe) between the multiply-adds of the following steps (FMA pipe), and the window starts with its DFT
// over t_hi.  Without this every warp of the SM decodes at the same time at the top of a window: the ALU pipe saturates
// and the FMA pipe idles (removing 64 of the 167 decode instructions, as an experiment, made cfg 3 7.6 % faster).  The
// copy of window i + 2 starts when all 16 warps have decoded window i + 1.  At RA = 16 (one gate per CTA) the stage
// saves no loads and exists for this alone (sc16 only: a complex64 window of 16384 does not fit beside the exchange).
// Measured: cfg 3 5.93 -> 5.81 ms (staged without early decode: 6.10), cfg 2 0.350 -> 0.346 ms, cfg 5 unchanged.
template <int RA, int Q, int DT, bool ST, bool PFE = true, int RQ = 0, int VDT = DT_CF32, bool IDC = false, bool ED = false>
__global__ void __launch_bounds__(kFusedThreads, 1) fused_kernel(const __grid_constant__ KParams P) {
    static_assert(!ED || (ST && Q == 1 && RQ == 0 && !IDC), "early decode: staged windows");
    static_assert(!ST || Q == 1, "the staged variant holds one whole window run in shared memory");
    static_assert(RQ == 0 || (RA == 16 && Q == 1 && DT == DT_CF32 && !ST && PFE), "ring mode: 16384-point complex64 windows");
    static_assert(!IDC || (RA == 16 && Q == 1 && DT == DT_CF32 && !ST && PFE && RQ == 0), "identity code: prefetching complex64 variant");
    constexpr int ESZ = DT == DT_CF32 ? 8 : 4;
    constexpr int NJ = 16 / RA;            // a' values per thread in pass A
    constexpr int G = 16 / RA;             // gates per CTA
    constexpr int LOGRA = ilog2(RA);
    // regions per "full" mbarrier.  Measured again on the early-decode kernels (profiles/r02b_experiments.md section 13):
    // RA = 16: 1 / 2 / 4 / 8 -> cfg 3 5.838 / 5.755 / 5.782 / 5.766 ms; RA = 8: 1 / 2 / 4 -> cfg 5 28.06 / 27.68 / 27.75 ms;
    // RA = 4: 1 / 2 / 4 -> cfg 2 0.3415 / 0.3367 / 0.3467 ms (round 1 had 4 at RA = 16 and 1 below)
    constexpr int FG = RA >= 4 ? 2 : 1;
    // A -> B1 exchange in 128-bit accesses, slot (a' * 32 + b) of 16 bytes = (y.re pair, y.im pair): half the shared-memory
    // instructions for the same wavefronts.  Measured: cfg 3 5.974 -> 5.923 ms, paper workload 12.63 -> 12.38 ms.  At
    // RA = 8 and 4 the register quads cost spills in the kernels of round 1 (cfg 5 28.2 -> 28.5 ms); in the early-decode
    // kernels they do not (cfg 5 28.13 -> 28.07 ms, cfg 2 0.3427 -> 0.3417 ms).
    constexpr bool X128 = RA >= 4;
    // Pass B2 as a decimation-in-time radix-32 (pairs = even / odd b) whose last stage -- the one across the two halves
    // of a register pair -- is fused with |X|^2 (bfly_power_halves), instead of the decimation-in-frequency form whose
    // first stage is across the halves: 420 instead of 448 FMA-pipe cycles per thread and window.  Measured: cfg 3
    // 5.833 -> 5.784 ms with the early-decode sc16 kernel at RA = 16; the other variants lose (register allocation:
    // the complex64 prefetch kernel spills 184 bytes, cfg 5 28.14 -> 28.35 ms, cfg 2 0.3429 -> 0.3447 ms), so only
    // that kernel takes this form.
    constexpr bool kB2Dit = ED && RA == 16 && DT == DT_SC16;
    constexpr int RB = kB2Dit ? kRegionBytesDit : kRegionBytes;    // region pitch
    constexpr int CTL = 16 * RB;                                    // control words behind the regions, then the stage
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = warp / RA, wa = warp % RA;       // pass A: warp `wa` of gate g;  pass B: (gate g, f_hi = wa)

    // ---- schedule: the launch's work items (tile, IPP), tile = (gate group, q), are numbered tile-major
    // and CTA c takes the contiguous run [c T / n, (c + 1) T / n) of the T = tiles * n_ipp items: equal
    // work for every CTA, accumulators flushed only where the run crosses into another tile.
    // (ring mode: n_groups = rounds, every CTA walks all rounds x IPPs)
    const long long T = RQ ? (long long)P.n_groups * P.n_ipp : (long long)P.n_groups * Q * P.n_ipp;
    const long long i0 = RQ ? 0 : (long long)blockIdx.x * T / gridDim.x;
    const long long i1 = RQ ? T : ((long long)blockIdx.x + 1) * T / gridDim.x;
    const int Rv = RQ ? P.R * RQ : P.R;            // gates the CTAs walk (ring mode: virtual gates)
    if (i0 >= i1) return;                          // uniform for the CTA; nothing allocated yet
    const int tile0 = (int)(i0 / P.n_ipp);
    const int p0 = (int)(i0 - (long long)tile0 * P.n_ipp);
    // tile -> gate group and residue
    auto group_of = [&](int t) { return RQ ? t * (int)gridDim.x + (int)blockIdx.x : (Q == 1 ? t : t % P.n_groups); };
    auto resid_of = [&](int t) { return Q == 1 ? 0 : t / P.n_groups; };
    // ---- ST: stage control.  mbar counts the bytes of one IPP's copy; cnt counts warps done reading it.
    const uint32_t mbar = smem_u32(smem + CTL);
    int *const cnt = reinterpret_cast<int *>(smem + CTL + 8);
    const unsigned char *const stage = smem + CTL + kStageCtlBytes;
    auto stage_issue = [&](int t, int pp) {                                // one thread: run of tile t, IPP pp
        const int tg = group_of(t);
        const int gates_here = (P.R - tg * G) < G ? (P.R - tg * G) : G;
        const uint32_t run_bytes = (uint32_t)((gates_here - 1) * P.stride + P.L) * ESZ;
        const long long roff = (long long)P.r0 + (long long)(tg * G) * P.stride;
        const unsigned char *src = reinterpret_cast<const unsigned char *>(P.V) + ((long long)pp * P.v_pitch + roff) * ESZ;
        const uint32_t mis = (uint32_t)(reinterpret_cast<uintptr_t>(src) & 15);
        const uint32_t bytes = (mis + run_bytes + 15u) & ~15u;
        mbar_arrive_expect_tx(mbar, bytes);
        for (uint32_t off = 0; off < bytes; off += 32768u)
            bulk_g2s(smem_u32(stage) + off, src - mis + off, (bytes - off) < 32768u ? (bytes - off) : 32768u, mbar);
    };
    // the first copy does not depend on anything earlier in the stream (the voltages are the caller's, or were copied
    // before the launch could start): it is started before the TMEM set-up and the griddepcontrol.wait below, so that its
    // DRAM latency hides under them
    if constexpr (ST) {
        if (tid == 0) {
            mbar_init(mbar, 1);
            *cnt = 0;
            fence_mbar_init();
            fence_proxy_async();
            stage_issue(tile0, p0);
        }
    }

    // ---- twiddles live in tensor memory: every thread re-reads only constants it wrote itself
    //   columns [4 e, 4 e + 4), e = (f - 1) NJ + jj:      pass A -> B1, W_Nk^{t_lo f} for the thread's two t_lo
    //   columns [64 + 4 c', ..):                           B1 -> B2,   W_1024^{b c'}, W_1024^{b (c' + 16)}, b = lane
    uint32_t *const tm_slot = reinterpret_cast<uint32_t *>(smem + CTL + 12);
    if (warp == 0) tmem_alloc_512(smem_u32(tm_slot));
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tm_base = *tm_slot;
    const uint32_t tm = tm_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 128);
    sfor<0, NJ>([&](auto jj_) {
        constexpr int jj = decltype(jj_)::value;
        const int ap = wa + RA * jj;
        sfor<1, RA>([&](auto f_) {
            constexpr int f = decltype(f_)::value;
            const float2 wr = __ldg(P.twA + ((ap * RA + f) * 2 + 0) * 32 + lane);
            const float2 wi = __ldg(P.twA + ((ap * RA + f) * 2 + 1) * 32 + lane);
            tmem_st4(tm + 4 * ((f - 1) * NJ + jj), wr.x, wr.y, wi.x, wi.y);
        });
    });
    sfor<0, 16>([&](auto c_) {
        constexpr int c = decltype(c_)::value;
        const float2 wr = __ldg(P.twB + (c * 2) * 32 + lane), wi = __ldg(P.twB + (c * 2 + 1) * 32 + lane);
        tmem_st4(tm + 64 + 4 * c, wr.x, wr.y, wi.x, wi.y);
    });
    tmem_wait_st();

    pdl_wait();   // everything above (TMEM, twiddles) may overlap the code pre-pass / decode pre-pass before us
    const bool bpsk = IDC || (P.Cbits != nullptr && __ldg(P.not_bpsk) != P.epoch);   // warp-uniform

    unsigned char *const region = smem + warp * RB;                        // this warp's pass-B region
    unsigned char *const gate_regions = smem + (g * RA) * RB;              // regions of this gate (pass A target)

    // Hand-over of the exchange regions without CTA-wide barriers.  full_mbar[region] (count RA): every pass-A
    // warp of the gate arrives after its last store into the region; the region's owner waits on it before
    // pass B1.  All warps store the regions in the same order f = 0 .. RA - 1, so the owners start pass B one
    // after the other and the stagger carries over to the next window: in steady state nobody waits.  At
    // RA >= 4 two neighbouring regions share one mbarrier (FG).
    // free_mbar[gate] (count RA): each owner arrives once it has read its region for the last time in a window
    // (B2 loads done); a pass-A warp waits on it before its first store of the next window (by then the last
    // owner is long past that point, and one probe per window is cheaper than one per region).
    const uint32_t free_base = smem_u32(smem + CTL + 16) + 8 * (g * RA);
    const uint32_t full_base = smem_u32(smem + CTL + 16 + 16 * 8) + 8 * (g * RA);  // + 8 f
    if (tid == 0) {
        for (int i = 0; i < 16; i++) {
            mbar_init(smem_u32(smem + CTL + 16 + 8 * i), RA);
            mbar_init(smem_u32(smem + CTL + 16 + 16 * 8 + 8 * i), RA);
        }
        if constexpr (RQ > 0) {
            for (int i = 0; i < 16; i++) reinterpret_cast<int *>(smem + CTL + kRingCtlOff)[i] = 0;
            mbar_init(smem_u32(smem + CTL + kRingCtlOff + 48), 1);
            mbar_init(smem_u32(smem + CTL + kRingCtlOff + 56), 1);
        }
        fence_mbar_init();
    }
    __syncthreads();
    if (RA > 1 && lane == 0) mbar_arrive(free_base);                      // phase 0: the regions start out free
    uint32_t parity = 0, free_parity = 0, full_parity = 0;
    int arrivals_target = 15;                                              // 16 warps per IPP, 0-based last

    // PF: the raw samples (one 32-bit word each) and the code word of the NEXT window are fetched while the last
    // butterfly stage of the current one retires its registers, so no warp sits on L2 latency at the top of a window
    constexpr bool PF = PFE && RA == 16 && Q == 1 && !ST;
    constexpr int WPS = DT == DT_SC16 ? 1 : 2;     // 32-bit words per sample
    uint32_t raw[PF ? 32 * WPS : 1], cw_pf = 0;
    auto pf_base = [&](int t, int pp) {            // this thread's first sample of (tile t, IPP pp)
        const int rr = group_of(t) * G + g;
        const long long off = (long long)P.r0 + (long long)(rr < P.R ? rr : P.R - 1) * P.stride;
        return reinterpret_cast<const uint32_t *>(P.V) + ((long long)pp * P.v_pitch + off + 64 * wa + lane) * WPS;
    };
    auto pf_load = [&](const uint32_t *b, auto i_) {   // sample i = 2 t_hi + o of the thread's window
        constexpr int i = decltype(i_)::value;
        if constexpr (DT == DT_SC16) {
            raw[i] = __ldg(b + (i >> 1) * 1024 + (i & 1) * 32);
        } else {
            const uint2 *a = reinterpret_cast<const uint2 *>(b) + (i >> 1) * 1024 + (i & 1) * 32;
            const uint2 v = RQ ? __ldcg(a) : __ldg(a);           // ring slots are rewritten during the launch: L2 only
            raw[2 * i] = v.x;
            raw[2 * i + 1] = v.y;
        }
    };
    if constexpr (PF) {
        if (bpsk) {
            const uint32_t *b = pf_base(tile0, p0);
            sfor<0, 32>([&](auto i_) { pf_load(b, i_); });
            if constexpr (!IDC) cw_pf = __ldg(P.Cbits + (long long)p0 * 512 + wa * 32 + lane);
        }
    }

    // ---- ring mode: producer side and the two hand-over counters per slot.  Arrivals are counted per CTA in shared
    // memory (by step & 3: the warps of a CTA are never more than a window or two apart) and the 16th warp of a step
    // passes the CTA's arrival on to the global counter, so a step completes at gridDim.x arrivals; the first warp
    // of a CTA that needs a step polls the global counter (one poller per CTA: every acquire load drops the SM's
    // L1) and publishes what it saw in shared memory for the other fifteen.
    const uint32_t ring_ctl = smem_u32(smem + CTL + kRingCtlOff);   // +0 ready cnt[4], +16 done cnt[4], +32 seen[2], +40 lock[2], +48 stage mbarrier[2]
    const bool r_staged = RQ > 0 && P.ring_stage != 0;
    const bool r_lean = r_staged && P.L == P.N && gridDim.x >= 16 && (P.c_pitch & 1) == 0;   // see ring_produce_lean_fn
    auto ring_arrive = [&](int which, int step) {       // which: 0 ready (after this warp's stores), 1 done (after its loads)
        __syncwarp();
        if (lane == 0) {
            const int old = atom_add_acq_rel_cta(ring_ctl + 16 * which + 4 * (int)(step & 3), 1);
            if ((old & 15) == 15) {
                red_release_add(P.ring_flags + 32 * (which * P.ring_depth + (int)(step % P.ring_depth)), 1);
                if (which == 0 && r_staged && step + 2 < (int)T) {     // every warp has read buffer step & 1 for the last time
                    fence_proxy_async();
                    if constexpr (RQ > 0) ring_stage_issue_fn<RQ, VDT>(&P, step + 2);
                }
            }
        }
    };
    auto ring_wait = [&](int which, int step) {         // until every CTA has arrived `which` for `step`
        if (lane == 0) {
            const uint32_t seen = ring_ctl + 32 + 4 * which, lock = ring_ctl + 40 + 4 * which;
            const int *f = P.ring_flags + 32 * (which * P.ring_depth + (int)(step % P.ring_depth));
            const int target = (int)(step / P.ring_depth + 1) * (int)gridDim.x;
            int spins = 0;
            while (ld_acquire_cta(seen) <= (int)step) {       // seen = number of leading steps known complete
                if (atom_cas_acquire_cta(lock, 0, 1) == 0) {
                    if (ld_acquire_cta(seen) <= (int)step) {
                        // bounded: if the grid were not fully resident (it is launched cooperatively, so it is) the
                        // wait would never end; after ~seconds give up, say so in the error word behind the
                        // counters, and run on
                        while (ld_acquire(f) < target) {
                            __nanosleep(32);
                            if (++spins > (1 << 22)) {
                                atomicExch(P.ring_flags + 64 * P.ring_depth, 1);
                                break;
                            }
                        }
                        st_release_cta(seen, (int)step + 1);
                    }
                    st_release_cta(lock, 0);
                } else {
                    __nanosleep(64);                          // another warp of the CTA is polling: stay out of the issue slots
                }
            }
        }
        __syncwarp();
    };
    // part 0: the first two gates of every thread, part 1: the rest + the arrival (-1: everything)
    auto ring_produce = [&](int sp, int part) {
        if constexpr (RQ > 0) {
            if (r_lean) ring_produce_lean_fn<RQ, VDT>(&P, sp, part);
            else ring_produce_fn<RQ, VDT>(&P, sp, part);
            if (part != 0) ring_arrive(0, sp);
        }
    };
    auto pf_ring = [&](int step) {           // this thread's first sample of its window in the slot of `step`
        return reinterpret_cast<const uint32_t *>(P.ring + ((size_t)(step % P.ring_depth) * gridDim.x + blockIdx.x) * (size_t)(1024 * RA) +
                                                  64 * wa + lane);
    };
    if constexpr (RQ > 0) {
        if (r_staged) {
            ring_stage_prologue_fn<RQ, VDT>(&P, (int)T);
            __syncthreads();
        }
        for (int sp = 0; sp < P.ring_ahead && sp < (int)T; sp++) ring_produce(sp, -1);
        if constexpr (PF) {                                          // the first window
            ring_wait(0, 0);
            const uint32_t *b = pf_ring(0);
            sfor<0, 32>([&](auto i_) { pf_load(b, i_); });
        }
    }

    // The walk over this CTA's work items, compiled once, or twice in the ED kernel: EDM = early decode in effect
    // (+-1 codes), where the decoded next window is carried from the tail of one window to the top of the next --
    // 64 registers that must not exist on the general-code path.
    auto run = [&](auto edm_) {
    constexpr bool EDM = decltype(edm_)::value;
    float2 nxr[EDM ? 16 : 1], nxi[EDM ? 16 : 1];
    // this thread's sample 0 of its gate's window of (tile t, IPP pp) in the stage (+ lane); its code words
    auto ed_src = [&](int t, int pp, uint32_t *cw) {
        const int rr = t * G + g < P.R ? t * G + g : P.R - 1;          // Q == 1: tile = gate group
        const uintptr_t a = reinterpret_cast<uintptr_t>(P.V) +
                            (uintptr_t)(((long long)pp * P.v_pitch + (long long)P.r0 + (long long)(t * G) * P.stride) * ESZ);
#pragma unroll
        for (int jj = 0; jj < NJ; jj++) cw[jj] = __ldg(P.Cbits + (long long)pp * 512 + (wa + RA * jj) * 32 + lane);
        return stage + ((long long)((a & 15) / ESZ) + (long long)(rr - t * G) * P.stride + lane) * ESZ;
    };
    // element e = jj RA + th of the thread: samples th 1024 + 64 (wa + RA jj) + lane (+ 32) -> nxr / nxi[e]
    auto ed_dec = [&](auto e_, const unsigned char *src, const uint32_t *cw) {
        constexpr int e = decltype(e_)::value, jj = e / RA, th = e % RA;
        if constexpr (EDM) {
            const int t0 = th * 1024 + 64 * (wa + RA * jj);
            const uint32_t m0 = bit_mask<2 * th>(cw[jj]), m1 = bit_mask<2 * th + 1>(cw[jj]);
            if constexpr (DT == DT_SC16) {
                const uint32_t *w = reinterpret_cast<const uint32_t *>(src) + t0;
                // some pairs through the conversion unit, spread evenly over the steps of the last butterfly stage, so that
                // both forms run side by side: every other pair (the steps free one even and one odd element each), or,
                // where pass B2 is the decimation-in-time form (sixteen steps, element brev4(step)), every fourth
                // (measured: 1/4, 1/2, 3/4 of the pairs -> cfg 3 5.742 / 5.767 / 5.843 ms, cfg 5 27.79 / 27.69 / 27.88 ms)
                if constexpr (kB2Dit ? (((e >> 2) & 3) == 3) : (e & 1)) sc16_pair_to_f32_xu(w[0], w[32], m0, m1, nxr[e], nxi[e]);
                else sc16_pair_to_f32(w[0], w[32], m0, m1, nxr[e], nxi[e]);
            } else {
                const uint2 *w = reinterpret_cast<const uint2 *>(src) + t0;
                const uint2 z0 = w[0], z1 = w[32];
                nxr[e] = make_float2(flip_sign(z0.x, m0), flip_sign(z1.x, m1));
                nxi[e] = make_float2(flip_sign(z0.y, m0), flip_sign(z1.y, m1));
            }
        }
    };
    auto ed_arrive = [&](bool issue, int t, int pp) {  // this warp is done with the stage; the 16th warp starts the next copy
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            const int old = atomicAdd(cnt, 1);
            if (old == arrivals_target && issue) {
                __threadfence_block();
                fence_proxy_async();
                stage_issue(t, pp);
            }
        }
        arrivals_target += 16;
    };
    if constexpr (EDM) {
        {                                              // the first window: nothing to hide it under
            uint32_t cw0[NJ];
            const unsigned char *s0 = ed_src(tile0, p0, cw0);
            mbar_wait(mbar, parity);
            parity ^= 1u;
            sfor<0, 16>([&](auto th_) { ed_dec(th_, s0, cw0); });
            int p1 = p0 + 1, t1 = tile0;
            if (p1 == P.n_ipp) { p1 = 0; t1++; }
            ed_arrive(i1 - i0 >= 2, t1, p1);
        }
    }

    int left = (int)(i1 - i0);                     // items still to do, this one included
    int p_lo = p0;
    // ring mode: a "tile" is a run of at most kRingFlushEvery pulses of one round -- two-level summation: fp32 sums of
    // many |X|^2 lose low bits to the running total, so no more than that many are summed in registers before they go
    // to S (the old scratch path flushed per batch of 10 as well)
    const int r_nch = RQ ? (P.n_ipp + kRingFlushEvery - 1) / kRingFlushEvery : 1;
    for (int tile = tile0; left > 0; tile++, p_lo = 0) {                   // the tiles this CTA's run touches
    int kround = tile;
    if constexpr (RQ > 0) {
        kround = tile / r_nch;
        p_lo = (tile - kround * r_nch) * kRingFlushEvery;
    }
    const int p_hi = RQ ? (P.n_ipp < p_lo + kRingFlushEvery ? P.n_ipp : p_lo + kRingFlushEvery)
                        : ((P.n_ipp - p_lo) < left ? P.n_ipp : p_lo + left);
    left -= p_hi - p_lo;
    const bool more_tiles = left > 0;
    const int gg = group_of(kround), q = resid_of(tile);
    const int r = gg * G + g;
    const int r_ld = r < Rv ? r : Rv - 1;          // ragged last group: recompute a valid gate, never flush it
    const long long gate_off = (long long)P.r0 + (long long)r_ld * P.stride;
    const long long run_off = (long long)P.r0 + (long long)(gg * G) * P.stride;   // first sample of the CTA's run
    // per last-stage butterfly of pass B2: packed pairs (even e, odd e) per k (bfly_power), or, kB2Dit, accS[k] =
    // (scalar of e'' = 2k, of e'' = 2k + 1) per output pair (e'', e'' + 16) (bfly_power_halves)
    float2 accS[8], accC[8];
#pragma unroll
    for (int j = 0; j < 8; j++) accS[j] = accC[j] = make_float2(0.f, 0.f);
    auto acc_ref = [&](float2 (&a)[8], auto e_) -> float & {
        constexpr int e = decltype(e_)::value;
        if constexpr (e & 1) return a[e / 2].y; else return a[e / 2].x;
    };
    for (int p = p_lo; p < p_hi; p++) {
        const bool has_next = p + 1 < p_hi || more_tiles;
        const int p_next = p + 1 < p_hi ? p + 1 : 0;
        const int tile_next = p + 1 < p_hi ? tile : tile + 1;
        int rs = 0;                                                  // ring mode: this step (the host keeps T below 2^20)
        if constexpr (RQ > 0) {
            rs = kround * P.n_ipp + p;
            if (r >= Rv) {                                           // a round with fewer virtual gates than CTAs: produce only
                const int sp = rs + P.ring_ahead;
                if (sp < (int)T) {
                    if (sp >= P.ring_depth) ring_wait(1, sp - P.ring_depth);
                    ring_produce(sp, -1);
                }
                ring_arrive(1, rs);
                if constexpr (PF) {                                  // (re-defines the prefetch registers, so that they
                    const uint32_t *b = pf_ring(rs);                 // need not survive the producer above)
                    sfor<0, 32>([&](auto i_) { pf_load(b, i_); });
                }
                continue;
            }
        }
        const float2 *Crow = P.C + (long long)p * P.L;
        const long long voff = (long long)p * P.v_pitch + gate_off;
        VSrc vs;
        vs.V = P.V; vs.voff = voff; vs.stage = stage; vs.sbase = 0;
        if constexpr (ST) {
            if constexpr (!EDM) {
                const uintptr_t a = reinterpret_cast<uintptr_t>(P.V) + (uintptr_t)(((long long)p * P.v_pitch + run_off) * ESZ);
                vs.sbase = (int)((a & 15) / ESZ) + (r_ld - gg * G) * P.stride;
                mbar_wait(mbar, parity);
                parity ^= 1u;
            }
        }
        float2 xr[16], xi[16];
        if constexpr (IDC) {
            // N > 16384, step 2: the window the last butterfly stage will fetch is asked into L2 now, a window's time
            // ahead -- its 128 KB come from the scratch in DRAM, and the register prefetch alone leaves them only the rest
            // of that stage to arrive (cfg 4 8.70 -> 8.55 ms; the paper workload, which misses L2 one time in ten, does
            // not gain: 12.12 -> 12.14 ms)
            if (has_next) {
                const int rr = group_of(tile_next) * G + g;
                const unsigned char *wb = reinterpret_cast<const unsigned char *>(P.V) +
                    ((long long)p_next * P.v_pitch + (long long)P.r0 + (long long)(rr < P.R ? rr : P.R - 1) * P.stride) * ESZ;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(wb + tid * 128));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(wb + 65536 + tid * 128));
            }
        }
        // ---- pass A: load + decode, x[jj*RA + t_hi] = (o = 0, o = 1)
        if constexpr (RQ > 0 || IDC) {                               // decoded already (prefetched from the ring / the scratch)
            sfor<0, RA>([&](auto th_) {
                constexpr int th = decltype(th_)::value;
                xr[th] = make_float2(__uint_as_float(raw[4 * th]), __uint_as_float(raw[4 * th + 2]));
                xi[th] = make_float2(__uint_as_float(raw[4 * th + 1]), __uint_as_float(raw[4 * th + 3]));
            });
        } else if constexpr (EDM) {                                  // decoded in the tail of the previous window
#pragma unroll
            for (int j = 0; j < 16; j++) { xr[j] = nxr[j]; xi[j] = nxi[j]; }
        } else if (PF && bpsk) {
            if constexpr (PF) {
                sfor<0, RA>([&](auto th_) {
                    constexpr int th = decltype(th_)::value;
                    const uint32_t m0 = bit_mask<2 * th>(cw_pf), m1 = bit_mask<2 * th + 1>(cw_pf);
                    if constexpr (DT == DT_SC16) {
                        sc16_pair_to_f32(raw[2 * th], raw[2 * th + 1], m0, m1, xr[th], xi[th]);
                    } else {                                     // +-1 code: flip the sign bits
                        xr[th] = make_float2(flip_sign(raw[4 * th], m0), flip_sign(raw[4 * th + 2], m1));
                        xi[th] = make_float2(flip_sign(raw[4 * th + 1], m0), flip_sign(raw[4 * th + 3], m1));
                    }
                });
            }
        } else if (bpsk) {
            sfor<0, NJ>([&](auto jj_) {
                constexpr int jj = decltype(jj_)::value;
                const int ap = wa + RA * jj;
                const int t_lo = 64 * ap + lane;
                uint32_t cw[Q];
#pragma unroll
                for (int j = 0; j < Q; j++) cw[j] = __ldg(P.Cbits + ((long long)p * Q + j) * 512 + ap * 32 + lane);
                sfor<0, RA>([&](auto th_) {
                    constexpr int th = decltype(th_)::value;
                    if constexpr (Q == 1) {
                        load_pair_bpsk<DT, th * 2, th * 2 + 1, ST>(vs, cw[0], th * 1024 + t_lo, th * 1024 + t_lo + 32,
                                                                    xr[jj * RA + th], xi[jj * RA + th]);
                    } else {
                        const float2 d0 = load_decoded_bpsk<Q, DT, th * 2, ST>(P, vs, cw, th * 1024 + t_lo, q);
                        const float2 d1 = load_decoded_bpsk<Q, DT, th * 2 + 1, ST>(P, vs, cw, th * 1024 + t_lo + 32, q);
                        xr[jj * RA + th] = make_float2(d0.x, d1.x);
                        xi[jj * RA + th] = make_float2(d0.y, d1.y);
                    }
                });
            });
        } else {
#pragma unroll
            for (int jj = 0; jj < NJ; jj++) {
                const int t_lo = 64 * (wa + RA * jj) + lane;
#pragma unroll
                for (int th = 0; th < RA; th++) {
                    const float2 d0 = load_decoded<Q, DT, ST>(P, vs, Crow, th * 1024 + t_lo, q);
                    const float2 d1 = load_decoded<Q, DT, ST>(P, vs, Crow, th * 1024 + t_lo + 32, q);
                    xr[jj * RA + th] = make_float2(d0.x, d1.x);
                    xi[jj * RA + th] = make_float2(d0.y, d1.y);
                }
            }
        }
        // DFT over t_hi, then y = X * W_Nk^{t_lo f_hi}; the first two twiddle pairs come in meanwhile
        constexpr int NE = NJ * (RA - 1);                        // twiddle entries of this thread (0 when RA == 1)
        float twe[8], two[8];                                    // even / odd groups of two entries
        if constexpr (NE > 0) tmem_ld8(tm, twe);
        sfor<0, NJ>([&](auto jj_) {
            constexpr int jj = decltype(jj_)::value;
            dft_packed<RA, jj * RA>(xr, xi);
        });
        if constexpr (RQ > 0) ring_arrive(1, rs);                   // this warp's loads of the slot have all returned
        if constexpr (ST) {
            // this warp has consumed its samples of IPP p; the last of the 16 warps starts the copy of IPP p + 1
            if constexpr (!EDM) ed_arrive(has_next, tile_next, p_next);
        }
        if constexpr (RA == 1) __syncwarp();
        else mbar_wait(free_base, free_parity);                          // every owner has read the previous window
        auto store_y = [&](auto jj_, auto f_, float2 yr, float2 yi) {   // y_{f}[t_lo] -> region of pass-B warp (g, f)
            constexpr int jj = decltype(jj_)::value, f = decltype(f_)::value;
            const int ap = wa + RA * jj;
            if constexpr (X128) {
                float4 *dst = reinterpret_cast<float4 *>(gate_regions + f * RB) + ap * 32 + lane;
                *dst = make_float4(yr.x, yr.y, yi.x, yi.y);
            } else {
                float2 *dst = reinterpret_cast<float2 *>(gate_regions + f * RB) + (ap * 2) * 32 + lane;
                dst[0] = yr;
                dst[32] = yi;
            }
            if constexpr (RA > 1 && jj == NJ - 1 && (f % FG == FG - 1 || f == RA - 1)) {   // last store into the regions of group f / FG
                __syncwarp();
                if (lane == 0) mbar_arrive(full_base + 8 * (f / FG));
            }
        };
        sfor<0, NJ>([&](auto jj_) {
            constexpr int jj = decltype(jj_)::value;
            store_y(jj_, std::integral_constant<int, 0>{}, xr[jj * RA], xi[jj * RA]);
        });
        sfor<0, (NE + 1) / 2>([&](auto g_) {
            constexpr int gi = decltype(g_)::value;
            float(&cur)[8] = (gi & 1) ? two : twe;
            float(&nxt)[8] = (gi & 1) ? twe : two;
            tmem_wait_ld8(cur);
            if constexpr (gi + 1 < (NE + 1) / 2) tmem_ld8(tm + 8 * (gi + 1), nxt);
            sfor<0, 2>([&](auto k_) {
                constexpr int k = decltype(k_)::value;
                constexpr int e = gi * 2 + k;
                if constexpr (e < NE) {
                    constexpr int jj = e % NJ, f = e / NJ + 1;
                    constexpr int ph = jj * RA + brev<LOGRA>(f);
                    const float2 wr = make_float2(cur[4 * k], cur[4 * k + 1]), wi = make_float2(cur[4 * k + 2], cur[4 * k + 3]);
                    store_y(std::integral_constant<int, jj>{}, std::integral_constant<int, f>{},
                            pfma(xr[ph], wr, pneg(pmul(xi[ph], wi))), pfma(xr[ph], wi, pmul(xi[ph], wr)));
                }
            });
        });
        if constexpr (RQ > 0) {
            // producer: the data registers are dead and the warp would only wait for the other warps' stores.  Slot sp % depth last held step sp - depth: every warp of the grid must have loaded it.
            const int sp = rs + P.ring_ahead;
            if (sp < (int)T && (wa & 1) == 0) {                   // even warps produce here, odd ones between B1 and B2:
                if (sp >= P.ring_depth) ring_wait(1, sp - P.ring_depth);   // one half's stores drain while the other half computes
                ring_produce(sp, -1);
            }
        }
        if constexpr (RA == 1) {
            __syncwarp();
        } else {
            free_parity ^= 1u;
            mbar_wait(full_base + 8 * (wa / FG), full_parity);                  // every pass-A warp has filled this warp's region
            full_parity ^= 1u;
        }

        // ---- pass B1: lane = b; decimation-in-time radix-32 over a; .x = even a, .y = odd a
        {
            if constexpr (X128) {
                const float4 *src = reinterpret_cast<const float4 *>(region) + lane;
#pragma unroll
                for (int ap = 0; ap < 16; ap++) {
                    const float4 v = src[ap * 32];
                    xr[ap] = make_float2(v.x, v.y);
                    xi[ap] = make_float2(v.z, v.w);
                }
            } else {
                const float2 *src = reinterpret_cast<const float2 *>(region) + lane;
#pragma unroll
                for (int ap = 0; ap < 16; ap++) {
                    xr[ap] = src[(ap * 2) * 32];
                    xi[ap] = src[(ap * 2 + 1) * 32];
                }
            }
        }
        __syncwarp();
        tmem_ld8(tm + 64, twe);
        dft_packed<16, 0>(xr, xi);                               // (E[c'], O[c']) at brev4(c')
        sfor<0, 8>([&](auto g_) {
            constexpr int gi = decltype(g_)::value;
            float(&cur)[8] = (gi & 1) ? two : twe;
            float(&nxt)[8] = (gi & 1) ? twe : two;
            tmem_wait_ld8(cur);
            if constexpr (gi + 1 < 8) tmem_ld8(tm + 64 + 8 * (gi + 1), nxt);
            sfor<0, 2>([&](auto k_) {
                constexpr int k = decltype(k_)::value;
                constexpr int c = gi * 2 + k;
                constexpr int ph = brev<4>(c);
                bfly_dit_halves<c>(xr[ph], xi[ph]);              // (.x, .y) = (c', c' + 16)
                const float2 wr = make_float2(cur[4 * k], cur[4 * k + 1]), wi = make_float2(cur[4 * k + 2], cur[4 * k + 3]);
                const float2 zr = pfma(xr[ph], wr, pneg(pmul(xi[ph], wi)));
                const float2 zi = pfma(xr[ph], wi, pmul(xi[ph], wr));
                if constexpr (kB2Dit) {                              // row (plane, c), column b = lane
                    float *dst = reinterpret_cast<float *>(region) + lane;
                    dst[c * 34] = zr.x;
                    dst[(c + 16) * 34] = zr.y;
                    dst[(32 + c) * 34] = zi.x;
                    dst[(32 + c + 16) * 34] = zi.y;
                } else {
                    float *dst = reinterpret_cast<float *>(region + (lane & 15) * (65 * 8) + (lane >> 4) * 4);
                    dst[(c) * 2] = zr.x;
                    dst[(c + 16) * 2] = zr.y;
                    dst[(32 + c) * 2] = zi.x;
                    dst[(32 + c + 16) * 2] = zi.y;
                }
            });
        });
        __syncwarp();
        if constexpr (RQ > 0) {                                  // producer, odd warps (data registers dead again)
            const int sp = rs + P.ring_ahead;
            if (sp < (int)T && (wa & 1) != 0) {
                if (sp >= P.ring_depth) ring_wait(1, sp - P.ring_depth);
                ring_produce(sp, -1);
            }
        }
        // ---- pass B2: lane = c; decimation-in-frequency radix-32 over b; .x = b, .y = b + 16
        auto b2_front = [&]() {
            if constexpr (kB2Dit) {                                  // lane = c: (.x, .y) = (b = 2 j, b = 2 j + 1)
                const float2 *sr = reinterpret_cast<const float2 *>(reinterpret_cast<const float *>(region) + lane * 34);
                const float2 *si = reinterpret_cast<const float2 *>(reinterpret_cast<const float *>(region) + (32 + lane) * 34);
#pragma unroll
                for (int j = 0; j < 16; j++) {
                    xr[j] = sr[j];
                    xi[j] = si[j];
                }
            } else {
                const float2 *src = reinterpret_cast<const float2 *>(region) + lane;
#pragma unroll
                for (int bb = 0; bb < 16; bb++) {
                    xr[bb] = src[bb * 65];
                    xi[bb] = src[bb * 65 + 32];
                }
            }
            if constexpr (RA > 1) {                                  // this warp's region may be overwritten again
                __syncwarp();
                if (lane == 0) mbar_arrive(free_base);
            }
            if constexpr (kB2Dit) {
                dft_packed<16, 0>(xr, xi);                           // (E[e''], O[e'']) at brev4(e'')
            } else {
                sfor<0, 16>([&](auto b_) {
                    constexpr int bb = decltype(b_)::value;
                    bfly_dif_halves<bb>(xr[bb], xi[bb]);             // (.x, .y) -> (even e, odd e) inputs
                });
                dft_packed16_head(xr, xi);
            }
        };
        if constexpr (EDM) {
            if (has_next) {                                      // pass B2 with the next window's decode in between
                uint32_t cwn[NJ];
                const unsigned char *sn = ed_src(tile_next, p_next, cwn);
                mbar_wait(mbar, parity);                         // its copy started a window ago
                parity ^= 1u;
                b2_front();                                      // same basic block as the decode below: the assembler may
                                                                 // start it as early as it finds registers
                if constexpr (kB2Dit) {
                    sfor<0, 16>([&](auto s_) {
                        constexpr int e2 = decltype(s_)::value, ph = brev<4>(e2);
                        bfly_power_halves<e2>(xr[ph], xi[ph], acc_ref(accS, s_), acc_ref(accC, s_));
                        ed_dec(std::integral_constant<int, ph>{}, sn, cwn);  // into the registers that just died
                    });
                } else {
                    sfor<0, 8>([&](auto k_) {
                        constexpr int k = decltype(k_)::value;
                        constexpr int ia = brev<4>(k), ib = brev<4>(k + 8);
                        bfly_power<2 * k>(xr[ia], xi[ia], xr[ib], xi[ib], accS[k], accC[k]);
                        ed_dec(std::integral_constant<int, ia>{}, sn, cwn);  // into the registers that just died
                        ed_dec(std::integral_constant<int, ib>{}, sn, cwn);
                    });
                }
                int p2 = p_next + 1, t2 = tile_next;
                if (p2 == P.n_ipp) { p2 = 0; t2++; }
                ed_arrive((p_hi - 1 - p) + left >= 2, t2, p2);
                continue;
            }
        }
        b2_front();
        const uint32_t *pf_next = nullptr;
        if constexpr (RQ > 0) {
            if (has_next) ring_wait(0, rs + 1);                  // the next window is in the ring (it has been for a while)
        }
        if constexpr (kB2Dit) {
            sfor<0, 16>([&](auto s_) {                           // last stage + |X|^2 + accumulate
                constexpr int e2 = decltype(s_)::value, ph = brev<4>(e2);
                bfly_power_halves<e2>(xr[ph], xi[ph], acc_ref(accS, s_), acc_ref(accC, s_));
                if constexpr (PF) {                              // four registers just died: two words of the next window
                    if constexpr (e2 == 0) {
                        if constexpr (RQ > 0) pf_next = pf_ring(has_next ? rs + 1 : rs);
                        else pf_next = has_next ? pf_base(tile_next, p_next) : pf_base(tile, p);
                    }
                    sfor<2 * e2, 2 * e2 + 2>([&](auto i_) { pf_load(pf_next, i_); });
                    if constexpr (e2 == 15) {
                        if constexpr (!IDC) {
                            if (bpsk) cw_pf = __ldg(P.Cbits + (long long)(has_next ? p_next : p) * 512 + wa * 32 + lane);
                        }
                    }
                }
            });
        } else
        sfor<0, 8>([&](auto k_) {                                // last stage + |X|^2 + accumulate
            constexpr int k = decltype(k_)::value;
            constexpr int ia = brev<4>(k), ib = brev<4>(k + 8);
            bfly_power<2 * k>(xr[ia], xi[ia], xr[ib], xi[ib], accS[k], accC[k]);
            if constexpr (PF) {                                  // eight registers just died: four words of the next window
                // unconditional (the last window fetches its own samples again): every word is redefined in every
                // window, so none of them stays live through passes A and B
                if constexpr (k == 0) {
                    if constexpr (RQ > 0) pf_next = pf_ring(has_next ? rs + 1 : rs);
                    else pf_next = has_next ? pf_base(tile_next, p_next) : pf_base(tile, p);
                }
                sfor<4 * k, 4 * k + 4>([&](auto i_) { pf_load(pf_next, i_); });
                if constexpr (k == 7) {
                    if constexpr (!IDC) {
                        if (bpsk) cw_pf = __ldg(P.Cbits + (long long)(has_next ? p_next : p) * 512 + wa * 32 + lane);
                    }
                }
            }
        });
        if constexpr (EDM) {
            // only the CTA's last window comes this way, but the compiler cannot know: without a definition here the
            // 64 carried registers would count as live through the whole loop body on this path, and be spilled
#pragma unroll
            for (int j = 0; j < 16; j++) nxr[j] = nxi[j] = make_float2(0.f, 0.f);
        }
    }
    // ---- flush: S_dev[r][q][f_hi = wa][e][c = lane]; other CTAs may hold the rest of this tile's IPPs
    if (r < Rv) {
        float *Srow = P.S + (((long long)r * Q + q) * RA + wa) * 1024 + lane;
        if constexpr (kB2Dit) {
            sfor<0, 16>([&](auto s_) {
                constexpr int e2 = decltype(s_)::value;
                const float c2 = acc_ref(accC, s_) * pow2w(e2), a = acc_ref(accS, s_);
                atomicAdd(Srow + e2 * 32, a + c2);
                atomicAdd(Srow + (e2 + 16) * 32, a - c2);
            });
        } else {
        float2 acc[16];                            // acc[j] = (S[e = 2 brev4(j)], S[e + 1]) at k_lo = lane + 32 e
        sfor<0, 8>([&](auto k_) {
            constexpr int k = decltype(k_)::value;
            const float2 c2 = pmul(accC[k], make_float2(pow2w(2 * k), pow2w(2 * k)));
            acc[brev<4>(k)] = padd(accS[k], c2);
            acc[brev<4>(k + 8)] = psub(accS[k], c2);
        });
        sfor<0, 16>([&](auto j_) {
            constexpr int j = decltype(j_)::value;
            constexpr int e = 2 * brev<4>(j);
            atomicAdd(Srow + e * 32, acc[j].x);
            atomicAdd(Srow + (e + 1) * 32, acc[j].y);
        });
        }
    }
    }
    };   // run
    if constexpr (ED) {
        if (bpsk) run(std::true_type{});
        else run(std::false_type{});
    } else {
        run(std::false_type{});
    }

    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc_512(tm_base);
}

// Finalize: natural bin order out, accumulators zeroed, one pass over S.  Per gate S_dev is an
// M x NC matrix, row j_in = q RAe + f_hi (M = Q RAe rows; fused layout: RAe = RA, NC = 1024; generic layout:
// RAe = 1, NC = Nk), and S_out[r][(f_hi Q + q) + M col] = S_dev[r][j_in][col]: a transposition.  A block moves a tile
// of all M rows x TC columns through shared memory (pitch M + 1), so both the reads and the writes are
// contiguous runs, and writes zeros back over what it has read.
__global__ void __launch_bounds__(256) finalize_kernel(float *__restrict__ Sdev, float *__restrict__ Sout, int log2Q,
                                                       int log2RAe, int NC, int TC) {
    extern __shared__ float tile[];
    const int log2M = log2Q + log2RAe, M = 1 << log2M, Q = 1 << log2Q, RAe = 1 << log2RAe;
    const long long gate = blockIdx.x;
    const int c0 = blockIdx.y * TC;
    float *X = Sdev + gate * (long long)M * NC;
    float *Y = Sout + gate * (long long)M * NC + (long long)c0 * M;
    const int n = M * TC;
    int log2TC = 0;
    while ((1 << log2TC) < TC) log2TC++;
    auto src_of = [&](int i) { return X + (long long)(i >> log2TC) * NC + c0 + (i & (TC - 1)); };
    for (int i0 = threadIdx.x; i0 < n; i0 += 8 * blockDim.x) {          // eight independent loads in flight per thread
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int i = i0 + u * blockDim.x;
            v[u] = i < n ? __ldcs(src_of(i)) : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int i = i0 + u * blockDim.x;
            const int j = i >> log2TC, c = i & (TC - 1);
            const int q = j >> log2RAe, f_hi = j & (RAe - 1);
            if (i < n) tile[c * (M + 1) + f_hi * Q + q] = v[u];
        }
    }
    __syncthreads();
    // zeros go back only now: a store to a line whose load is still in flight stalls the memory pipeline
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        Y[i] = tile[i + (i >> log2M)];
        *src_of(i) = 0.0f;
    }
}

// Finalize with the post-integration products folded into the write-out ("a row-wise reduction
// that fuses into finalize"): finalize_kernel's transposition, same grid (gate, column tile), and while a tile's bins
// pass through the CTA in natural order they are also (optionally) divided by n_ipp and written to P_out
// (Eq. 8, centred or not) and fed to the arg maxima / float64 sum of plspec_profile (profile_kernel has
// the definitions).  S is read once and S_out, P_out written once: no extra pass.  The CTAs of a gate meet in a
// 32-byte workspace per gate (zeroed by the caller): the arg maxima as 64-bit keys (value bits << 32 | ~bin: S >= 0,
// so the float's bit pattern orders like its value, and the lowest bin wins a tie) through atomicMax, the sum through a
// float64 atomicAdd; products_tail_kernel then takes the bins near the lines out of the sum again and writes the five
// per-gate numbers.
struct ProductsWork { unsigned long long up, dn; double sum; unsigned long long pad; };

__global__ void __launch_bounds__(256) finalize_products_kernel(float *__restrict__ Sdev, float *__restrict__ Sout, int log2Q,
                                                                int log2RAe, int NC, int TC, float *__restrict__ Pout, int centred,
                                                                int n_ipp, int k_min, ProductsWork *__restrict__ work) {
    extern __shared__ float tile[];
    __shared__ unsigned long long sb[2][8];
    __shared__ double ssum[8];
    const int log2M = log2Q + log2RAe, M = 1 << log2M, Q = 1 << log2Q, RAe = 1 << log2RAe;
    const long long gate = blockIdx.x;
    const int c0 = blockIdx.y * TC;
    const int N = M * NC, n = M * TC;
    float *X = Sdev + gate * (long long)N;
    float *Yrow = Sout + gate * (long long)N;
    float *Prow = Pout ? Pout + gate * (long long)N : nullptr;
    int log2TC = 0;
    while ((1 << log2TC) < TC) log2TC++;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lo = k_min, hi = N - k_min, mid = N / 2, half = centred ? N / 2 : 0;
    const float dn_ipp = (float)n_ipp;
    auto src_of = [&](int i) { return X + (long long)(i >> log2TC) * NC + c0 + (i & (TC - 1)); };
    for (int i0 = tid; i0 < n; i0 += 8 * 256) {                         // eight independent loads in flight per thread
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int i = i0 + u * 256;
            v[u] = i < n ? __ldcs(src_of(i)) : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < 8; u++) {
            const int i = i0 + u * 256;
            const int j = i >> log2TC, c = i & (TC - 1);
            const int q = j >> log2RAe, f_hi = j & (RAe - 1);
            if (i < n) tile[c * (M + 1) + f_hi * Q + q] = v[u];
        }
    }
    __syncthreads();
    unsigned long long up = 0, dn = 0;                                 // key 0 = "no bin": below every real key
    // a thread meets at most 16 bins: their sum in float32 (sequential: <= 15 roundings of 2^-24 relative, against the
    // 1e-6 the noise floor is good to), the CTA's and the gate's sums in float64 -- float64 adds are scarce on this part
    float facc = 0.f;
    const int f0 = c0 * M;                                              // first natural bin of this tile
    for (int i = tid; i < n; i += 256) {
        const float x = tile[i + (i >> log2M)];
        const int f = f0 + i;
        Yrow[f] = x;
        *src_of(i) = 0.0f;
        if (Prow) Prow[(f + half) & (N - 1)] = __fdiv_rn(x, dn_ipp);
        if (work && f >= lo && f <= hi && f != mid) {
            const unsigned long long key = ((unsigned long long)__float_as_uint(x) << 32) | (unsigned)(~f);
            if (f < mid) up = key > up ? key : up; else dn = key > dn ? key : dn;
            facc += x;
        }
    }
    if (!work) return;
    double acc = (double)facc;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        const unsigned long long u = __shfl_xor_sync(0xffffffffu, up, o), d = __shfl_xor_sync(0xffffffffu, dn, o);
        up = u > up ? u : up; dn = d > dn ? d : dn;
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
    }
    if (lane == 0) { sb[0][warp] = up; sb[1][warp] = dn; ssum[warp] = acc; }
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < 8; w++) {
            up = sb[0][w] > up ? sb[0][w] : up; dn = sb[1][w] > dn ? sb[1][w] : dn;
            acc += ssum[w];
        }
        if (up) atomicMax(&work[gate].up, up);
        if (dn) atomicMax(&work[gate].dn, dn);
        atomicAdd(&work[gate].sum, acc);
    }
}

// one warp per gate: the five numbers of plspec_profile from the workspace and the finished row of S_out
__global__ void __launch_bounds__(128) products_tail_kernel(const float *__restrict__ Sout, const ProductsWork *__restrict__ work,
                                                            int R, int N, int n_ipp, int k_min, int guard, int *__restrict__ k_up,
                                                            float *__restrict__ p_up, int *__restrict__ k_dn,
                                                            float *__restrict__ p_dn, float *__restrict__ noise) {
    const int gate = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (gate >= R) return;
    const float *row = Sout + (long long)gate * N;
    const int lo = k_min, hi = N - k_min, mid = N / 2;
    const ProductsWork w = work[gate];
    const int ku = (int)~(unsigned)(w.up & 0xffffffffu), kd = (int)~(unsigned)(w.dn & 0xffffffffu);
    const int g = guard < N ? guard : N, wlen = 2 * g + 1;
    double ex = 0.0;
    int nex = 0;
    for (int j = lane; j < 2 * wlen; j += 32) {                         // the bins within `guard` of either line, each once
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
    if (lane == 0) {
        k_up[gate] = ku; k_dn[gate] = kd;
        p_up[gate] = __uint_as_float((unsigned)(w.up >> 32)) / (float)n_ipp;
        p_dn[gate] = __uint_as_float((unsigned)(w.dn >> 32)) / (float)n_ipp;
        const int cnt = (hi - lo) - nex;                               // hi - lo + 1 searched bins less N/2
        noise[gate] = cnt > 0 ? (float)((w.sum - ex) / (double)cnt / (double)n_ipp) : 0.f;
    }
}

}  // namespace plspec
