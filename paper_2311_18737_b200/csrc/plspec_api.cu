// plspec_api.cu -- C ABI (include/plspec.h), handle, validation, launch logic and the
// multi-stream host loop.  No CPU compute path exists: every
// step of decode / FFT / power / accumulate runs in the kernels of plspec_kernels.cuh.
#include "../../include/plspec.h"
#include "plspec_kernels.cuh"
#include "plspec_fused.cuh"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace plspec;

namespace {

constexpr int kSlots = 3;            // host->device staging ring depth
constexpr int kMaxNk = 16384;        // largest window one SM holds (fused and generic kernels)
constexpr int kMaxRanges = 8;        // gate ranges of the overlapped write-out (plspec_finalize to a host buffer)
constexpr size_t kTailMaxBytes = (size_t)256 << 20;   // device staging of the deferred IPPs of a host-buffer call

struct Slot {
    void   *V = nullptr;             // [batch][span] voltages (storage dtype)
    float2 *C = nullptr;             // [batch][L]
    cudaEvent_t ready = nullptr;     // copies into the slot finished   (recorded on copy stream)
    cudaEvent_t freed = nullptr;     // kernel reading the slot finished (recorded on compute stream)
    bool used = false;
};

// Codes of one launch as the kernels want them: the one code of shared-code mode spread over n_ipp rows, and the
// bit-packed signs of +-1 codes.  Two instances per handle: the launch in flight, and the deferred tail (below).
struct CodePrep {
    float2 *crep = nullptr;          // shared-code mode: [n_ipp][L]
    long long crep_elems = 0;
    uint32_t *cbits = nullptr;       // [n_ipp][Q][512] packed code signs (BPSK fast path)
    long long cbits_words = 0;
    int flag = 0;                    // index of this instance's word in plspec_ctx::not_bpsk
    // result of prepare_codes
    const float2 *C = nullptr;       // codes[n_ipp][L] the kernels read
    bool packed = false;             // cbits holds this launch's signs; the flag word says whether they apply
    int epoch = 1;
};

// Host-buffer calls (a0): the last IPPs of the latest plspec_accumulate are copied to the device but NOT transformed
// yet.  If plspec_finalize comes next they are transformed one gate range after the other, and each range's spectra
// are un-permuted and copied out while the next range is still being transformed (the write-out overlaps the
// compute instead of following it); if another plspec_accumulate comes first they are transformed then, over all
// gates at once, like every other batch.
struct Tail {
    void   *V = nullptr;             // [n_ipp][span]
    float2 *C = nullptr;             // [n_ipp][L] (one row in shared-code mode)
    size_t v_bytes = 0, c_bytes = 0; // capacities
    int n_ipp = 0;
    bool pending = false;
    cudaEvent_t ready = nullptr;     // copies landed (copy stream)
    cudaEvent_t done = nullptr;      // kernels that read the buffers finished
    bool used = false;
    CodePrep cp;
};

}  // namespace

struct plspec_ctx {
    int N, L, R, r0, stride, ipp_len, dtype;
    int span;                        // (R-1)*stride + L samples needed from r0 on
    int device = 0, n_sm = 0;
    // kernel selection
    int kind = 2;                    // 1 generic, 2 fused
    int Nk = 0, Q = 1, RA = 1;   // N = Q * Nk, Nk = 1024 * RA (fused)
    int gates_per_cta = 1, n_groups = 0;
    int opt_kernel = 0, opt_chunks = 0, opt_batch = 0, opt_bpsk = 1, opt_stage = 1, opt_split = 1, opt_shared_code = 0;
    int opt_defer = 1;
    // N > 16384, ring mode (PLSPEC_OPT_SPLIT = 2, fused kernel only): one cooperative launch of the Q == 1 fused kernel whose CTAs
    // decode + butterfly every window once into a ring that stays in L2 and transform it from there
    bool ring_mode = false;
    const void *kfunc_ring = nullptr;    // fused_kernel<16, 1, CF32, false, true, Q, dtype>
    float2 *ring = nullptr;              // [ring_depth][ring_ctas][Nk]
    int *ring_flags = nullptr;           // [2][ring_depth] x 32 ints
    int ring_depth = 0, ring_ctas = 0;   // as allocated
    int opt_ring_depth = 3, opt_ring_ahead = 2;
    // split path for N > 16384 (PLSPEC_OPT_SPLIT = 1, the default): decode + outer butterfly once into `xq` (device scratch), then
    // the Q == 1 fused kernel over R * Q virtual gates of length Nk
    bool split = false;
    const void *kfunc_split = nullptr;   // fused_kernel<16, 1, CF32, false>
    float2 *xq = nullptr;                // [batch][R][Q][Nk]
    long long xq_ipps = 0;               // IPPs the scratch holds
    bool staged = false;             // fused kernel reads voltages through the shared-memory stage
    int block = 0;
    size_t smem = 0;
    int slots_per_wave = 0;          // n_sm * resident CTAs per SM
    const void *kfunc = nullptr;
    // device state
    float  *S = nullptr;             // [R][Q][Nk]
    float  *S_tmp = nullptr;         // un-permute target when S_out is a host pointer
    void   *prod_work = nullptr;     // plspec_finalize_products: ProductsWork[R]
    float2 *twA = nullptr, *twB = nullptr, *twN = nullptr;
    CodePrep cp;                     // codes of the launch in flight
    int *not_bpsk = nullptr;         // device flags written by pack_codes_kernel: [0] cp, [2] tail.cp
    int epoch = 0;                   // number of the last code pre-pass
    // host pipeline
    cudaStream_t copy_stream = nullptr;
    Slot slot[kSlots];
    int slot_batch = 0;              // IPPs each slot can hold
    int next_slot = 0;
    Tail tail;
    cudaStream_t d2h_stream = nullptr;
    cudaEvent_t range_done[kMaxRanges] = {};
    // ordering
    cudaEvent_t work_done = nullptr;
    cudaStream_t last_stream = nullptr;
    bool have_work = false;
    // bookkeeping
    int last_cuda = 0;
    plspec_stats_t stats;
};

namespace {

#define PL_CUDA(h, call)                                                   \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) {                                          \
            if (h) (h)->last_cuda = (int)e__;                              \
            (void)cudaGetLastError();                                      \
            return PLSPEC_ERR_CUDA;                                        \
        }                                                                  \
    } while (0)

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// SM count of the current device (the handle-free calls size their grids with it); 0 on error
int device_sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return n;
}

template <int RA, int Q, bool ST, bool PFE = true, bool ED = false>
const void *fused_ptr(int dt) {
    return dt == DT_CF32 ? (const void *)fused_kernel<RA, Q, DT_CF32, ST, PFE, 0, DT_CF32, false, ED>
                         : (const void *)fused_kernel<RA, Q, DT_SC16, ST, PFE, 0, DT_CF32, false, ED>;
}
// the outer radix Q > 1 only occurs with the largest inner size (Nk = 16384, RA = 16).  `prefetch`: the direct-load
// kernel at Nk = 16384 may fetch the whole next window ahead of time (only safe when code_len == N)
const void *fused_lookup(int RA, int Q, int dt, bool st, bool prefetch, bool early_decode) {
    if (Q == 1) {
        if (early_decode && st) {
            switch (RA) {
                case 1:  return fused_ptr<1, 1, true, true, true>(dt);
                case 2:  return fused_ptr<2, 1, true, true, true>(dt);
                case 4:  return fused_ptr<4, 1, true, true, true>(dt);
                case 8:  return fused_ptr<8, 1, true, true, true>(dt);
                case 16: return fused_ptr<16, 1, true, true, true>(dt);
            }
        }
        if (RA == 16 && !st && !prefetch) return fused_ptr<16, 1, false, false>(dt);
        switch (RA) {
            case 1:  return st ? fused_ptr<1, 1, true>(dt) : fused_ptr<1, 1, false>(dt);
            case 2:  return st ? fused_ptr<2, 1, true>(dt) : fused_ptr<2, 1, false>(dt);
            case 4:  return st ? fused_ptr<4, 1, true>(dt) : fused_ptr<4, 1, false>(dt);
            case 8:  return st ? fused_ptr<8, 1, true>(dt) : fused_ptr<8, 1, false>(dt);
            case 16: return st ? fused_ptr<16, 1, true>(dt) : fused_ptr<16, 1, false>(dt);
        }
    } else if (RA == 16 && !st) {
        if (Q == 2) return fused_ptr<16, 2, false>(dt);
        if (Q == 4) return fused_ptr<16, 4, false>(dt);
    }
    return nullptr;
}

// Resolve kernel kind / geometry from N and the options; (re)build what depends on it.
int select_kernel(plspec_ctx *h) {
    int kind = h->opt_kernel ? h->opt_kernel : (h->N >= 1024 ? 2 : 1);
    if (kind == 2 && h->N < 1024) return PLSPEC_ERR_UNSUPPORTED;
    h->kind = kind;
    h->Nk = h->N < kMaxNk ? h->N : kMaxNk;
    h->Q = h->N / h->Nk;
    const int dt = h->dtype == PLSPEC_SC16 ? DT_SC16 : DT_CF32;
    if (kind == 2) {
        h->RA = h->Nk / 1024;
        h->gates_per_cta = 16 / h->RA;
        h->block = kFusedThreads;
        h->smem = (size_t)kStageOff;                       // exchange regions + control words
        // staged variant: the run of samples one CTA's gates touch per IPP must fit beside the exchange regions
        const long long esz = dt == DT_SC16 ? 4 : 8;
        const long long run = ((long long)(h->gates_per_cta - 1) * h->stride + h->L) * esz;
        // opt_stage: 1 = where the run is shared by several gates of the CTA (measured: with one gate per CTA
        // the stage only adds shared-memory traffic), 2 = wherever it fits, 0 = never
        h->staged = h->opt_stage && h->Q == 1 && run + 32 <= (long long)kStageMaxBytes &&
                    (h->gates_per_cta > 1 || h->opt_stage == 2);
        // early decode (plspec_fused.cuh, ED; the default, opt_stage == 1): with a full-length code the next window is
        // decoded from the stage inside the last butterfly stage of the current one; sc16 windows of 16384 go through
        // the stage for that reason alone
        // (that kernel's exchange regions are larger: pass B2 in its decimation-in-time form, kDitExtraBytes)
        const bool dit = h->opt_stage == 1 && h->RA == 16 && h->Q == 1 && dt == DT_SC16 && h->L == h->N &&
                         run + 32 <= (long long)kStageMaxBytes - kDitExtraBytes;
        if (dit) h->staged = true;
        const bool early = h->opt_stage == 1 && h->staged && h->L == h->N;
        if (h->staged) h->smem = (size_t)kStageOff + (dit ? (size_t)kDitExtraBytes : 0) + (size_t)((run + 15) / 16 * 16 + 16);
        h->kfunc = fused_lookup(h->RA, h->Q, dt, h->staged, h->L == h->N, early);
        h->split = h->opt_split == 1 && h->Q > 1;
        h->ring_mode = h->opt_split == 2 && h->Q > 1;
        if (h->ring_mode) {
            h->kfunc_ring = h->Q == 2 ? (dt == DT_CF32 ? (const void *)fused_kernel<16, 1, DT_CF32, false, true, 2, DT_CF32>
                                                       : (const void *)fused_kernel<16, 1, DT_CF32, false, true, 2, DT_SC16>)
                                      : (dt == DT_CF32 ? (const void *)fused_kernel<16, 1, DT_CF32, false, true, 4, DT_CF32>
                                                       : (const void *)fused_kernel<16, 1, DT_CF32, false, true, 4, DT_SC16>);
            PL_CUDA(h, cudaFuncSetAttribute(h->kfunc_ring, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));
            int occ_ring = 0;
            PL_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_ring, h->kfunc_ring, kFusedThreads, (size_t)kStageOff));
            if (occ_ring < 1) return PLSPEC_ERR_UNSUPPORTED;
        }
        if (h->split) {
            // scratch windows are whole (Nk samples each) and decoded already: prefetching variant, identity code
            h->kfunc_split = (const void *)fused_kernel<16, 1, DT_CF32, false, true, 0, DT_CF32, true>;
            PL_CUDA(h, cudaFuncSetAttribute(h->kfunc_split, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStageOff));
        }
    } else {
        h->RA = 0;
        h->split = false;
        h->ring_mode = false;
        h->gates_per_cta = 1;
        h->block = h->Nk / 2 < 32 ? 32 : (h->Nk / 2 > 512 ? 512 : h->Nk / 2);
        h->smem = (size_t)h->Nk * (sizeof(float2) + sizeof(float));
        h->kfunc = dt == DT_CF32 ? (const void *)generic_kernel<DT_CF32> : (const void *)generic_kernel<DT_SC16>;
    }
    if (!h->kfunc) return PLSPEC_ERR_UNSUPPORTED;
    PL_CUDA(h, cudaFuncSetAttribute(h->kfunc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem));
    int occ = 0;
    PL_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->kfunc, h->block, h->smem));
    if (occ < 1) return PLSPEC_ERR_UNSUPPORTED;
    h->slots_per_wave = occ * h->n_sm;
    h->n_groups = (h->R + h->gates_per_cta - 1) / h->gates_per_cta;
    h->stats.kernel_kind = kind;
    return PLSPEC_OK;
}

int launch_split(plspec_ctx *h, const void *dV, const float2 *dC, long long v_pitch, int r0, int n_ipp, int g_lo,
                 int g_cnt, cudaStream_t stream);
int launch_ring(plspec_ctx *h, const void *dV, const float2 *dC, long long v_pitch, int r0, int n_ipp, int g_lo,
                int g_cnt, cudaStream_t stream);

// The fused kernel is launched with programmatic stream serialisation: its prologue (TMEM allocation, twiddle
// tables) overlaps the tail of whatever precedes it in the stream; it calls griddepcontrol.wait before it reads
// or writes anything earlier work produces.
cudaError_t launch_fused(const void *func, unsigned grid, unsigned block, void **args, size_t smem, cudaStream_t stream,
                         bool pdl) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelExC(&cfg, func, args);
}

// PLSPEC_OPT_SHARED_CODE: the one code of the call is spread over n_ipp rows of a device buffer, so that every
// kernel keeps its one-code-per-IPP indexing (what the mode saves is the caller's memory and the H2D copy).
__global__ void replicate_code_kernel(const float2 *__restrict__ code, float2 *__restrict__ rows, int L, long long total) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
        rows[i] = __ldg(code + (int)(i % L));
}

// Step 1 of a launch: bring the codes of n_ipp pulses into the form the kernels read (cp.C, cp.cbits).
int prepare_codes(plspec_ctx *h, CodePrep &cp, const float2 *dC, int n_ipp, cudaStream_t stream) {
    if (h->kind == 2 && (h->ring_mode || h->split)) {    // these paths read the codes as given (row pitch 0 or L)
        cp.C = dC; cp.packed = false; cp.epoch = 1;
        return PLSPEC_OK;
    }
    if (h->opt_shared_code) {
        const long long total = (long long)n_ipp * h->L;
        if (total > cp.crep_elems) {
            if (cp.crep) cudaFree(cp.crep);
            cp.crep = nullptr; cp.crep_elems = 0;
            if (cudaMalloc((void **)&cp.crep, sizeof(float2) * (size_t)total) != cudaSuccess) {
                (void)cudaGetLastError();
                return PLSPEC_ERR_ALLOC;
            }
            cp.crep_elems = total;
        }
        replicate_code_kernel<<<h->n_sm * 4, 256, 0, stream>>>(dC, cp.crep, h->L, total);
        PL_CUDA(h, cudaGetLastError());
        h->stats.kernel_launches++;
        dC = cp.crep;
    }
    cp.C = dC;
    cp.packed = false;
    cp.epoch = 1;
    if (h->kind == 2 && !h->split && h->opt_bpsk && h->L == h->N) {
        // code pre-pass: pack the signs of real +-1 codes (1 bit / sample instead of 8 bytes); the fused
        // kernel falls back to the general complex decode when the flag says the codes are anything else
        const long long words = (long long)n_ipp * h->Q * 512;
        if (words > cp.cbits_words) {
            if (cp.cbits) cudaFree(cp.cbits);
            cp.cbits = nullptr; cp.cbits_words = 0;
            if (cudaMalloc((void **)&cp.cbits, sizeof(uint32_t) * (size_t)words) != cudaSuccess) {
                (void)cudaGetLastError();
                return PLSPEC_ERR_ALLOC;
            }
            cp.cbits_words = words;
        }
        h->epoch = h->epoch == 0x7fffffff ? 1 : h->epoch + 1;
        cp.epoch = h->epoch;
        pack_codes_kernel<<<(unsigned)((words + 255) / 256), 256, 0, stream>>>(dC, cp.cbits, h->not_bpsk + cp.flag, cp.epoch,
                                                                              h->L, h->Nk, h->RA, h->Q, words);
        PL_CUDA(h, cudaGetLastError());
        h->stats.kernel_launches++;
        cp.packed = true;
    }
    return PLSPEC_OK;
}

// Step 2 of a launch: decode + FFT + power + accumulate of n_ipp pulses for the gates [g_lo, g_lo + g_cnt) into
// their rows of S_dev.  g_lo is a multiple of the fused kernel's gates per CTA.  r0 = sample of gate 0 in a row of dV.
int launch_gates(plspec_ctx *h, const CodePrep &cp, const void *dV, long long v_pitch, int r0, int n_ipp, int g_lo, int g_cnt,
                 cudaStream_t stream) {
    if (h->kind == 2 && h->ring_mode) return launch_ring(h, dV, cp.C, v_pitch, r0, n_ipp, g_lo, g_cnt, stream);
    if (h->kind == 2 && h->split) return launch_split(h, dV, cp.C, v_pitch, r0, n_ipp, g_lo, g_cnt, stream);
    const int n_groups = (g_cnt + h->gates_per_cta - 1) / h->gates_per_cta;
    KParams P{};
    P.V = dV; P.C = cp.C; P.S = h->S + (size_t)g_lo * (size_t)h->N;
    P.twA = h->twA; P.twB = h->twB; P.twN = h->twN;
    P.v_pitch = v_pitch;
    P.N = h->N; P.Nk = h->Nk; P.Q = h->Q; P.log2Nk = ilog2(h->Nk);
    P.L = h->L; P.R = g_cnt; P.r0 = r0 + g_lo * h->stride; P.stride = h->stride;
    P.n_groups = n_groups;
    P.n_ipp = n_ipp;
    P.Cbits = cp.packed ? cp.cbits : nullptr;
    P.not_bpsk = cp.packed ? h->not_bpsk + cp.flag : nullptr;
    P.epoch = cp.epoch;
    long long tiles;
    if (h->kind == 2) {
        // fused kernel: flattened schedule.  auto = one CTA per resident slot, each an equal run of
        // (tile, IPP) items; explicit chunks = that many equal IPP runs per tile, one CTA each
        const long long items = (long long)n_groups * h->Q * n_ipp;
        if (h->opt_chunks > 0) {
            P.n_chunks = h->opt_chunks < n_ipp ? h->opt_chunks : n_ipp;
            tiles = (long long)n_groups * h->Q * P.n_chunks;
        } else {
            P.n_chunks = 0;
            tiles = items < h->slots_per_wave ? items : h->slots_per_wave;
        }
        P.use_atomic = 1;
    } else {
        // generic kernel: one CTA per (gate, residue, IPP chunk); chunks picked for whole waves
        int c = h->opt_chunks > 0 ? (h->opt_chunks < n_ipp ? h->opt_chunks : n_ipp) : 1;
        if (h->opt_chunks <= 0) {
            const long long base = (long long)g_cnt * h->Q;
            double best_score = -1.0;
            for (int k = 1; k <= n_ipp && k <= 64; k++) {
                const long long t = base * k, waves = (t + h->slots_per_wave - 1) / h->slots_per_wave;
                const double eff = (double)t / (double)(waves * h->slots_per_wave), per = (double)n_ipp / k;
                const double score = eff * per / (per + 0.5);              // a flush costs ~half a window
                if (score > best_score + 1e-9) { best_score = score; c = k; }
            }
        }
        P.n_chunks = c;
        P.use_atomic = c > 1 ? 1 : 0;
        tiles = (long long)g_cnt * h->Q * c;
    }
    h->stats.ipp_chunks_last = P.n_chunks;
    if (tiles > 0x7fffffffLL) return PLSPEC_ERR_UNSUPPORTED;
    void *args[] = {&P};
    PL_CUDA(h, launch_fused(h->kfunc, (unsigned)tiles, (unsigned)h->block, args, h->smem, stream, h->kind == 2));
    h->stats.kernel_launches++;
    return PLSPEC_OK;
}

int launch_accumulate(plspec_ctx *h, const void *dV, const float2 *dC, long long v_pitch, int r0,
                      int n_ipp, cudaStream_t stream) {
    const int rc = prepare_codes(h, h->cp, dC, n_ipp, stream);
    if (rc != PLSPEC_OK) return rc;
    return launch_gates(h, h->cp, dV, v_pitch, r0, n_ipp, 0, h->R, stream);
}

// N > 16384, ring mode (plspec_fused.cuh): ONE cooperative launch per <= 2^20 steps.  gridDim.x = the largest
// multiple of Q that is resident at once (and no more than the launch has virtual gates); round k gives CTA c the
// virtual gate k gridDim.x + c; the ring holds `depth` steps of gridDim.x residues (depth x 148 x 128 KB = 76 MB at
// depth 4: inside the 126 MB L2 together with the voltages the producers read).
int launch_ring(plspec_ctx *h, const void *dV, const float2 *dC, long long v_pitch, int r0, int n_ipp, int g_lo,
                int g_cnt, cudaStream_t stream) {
    const int Q = h->Q;
    const int cta_max = (h->n_sm / Q) * Q;
    if (cta_max < Q) return PLSPEC_ERR_UNSUPPORTED;
    const int depth = h->opt_ring_depth, ahead = h->opt_ring_ahead < depth ? h->opt_ring_ahead : depth - 1;
    if (!h->ring || h->ring_depth != depth || h->ring_ctas != cta_max) {
        if (h->ring) cudaFree(h->ring);                   // waits for the device
        if (h->ring_flags) cudaFree(h->ring_flags);
        h->ring = nullptr; h->ring_flags = nullptr; h->ring_depth = 0;
        if (cudaMalloc((void **)&h->ring, (size_t)depth * cta_max * (size_t)h->Nk * sizeof(float2)) != cudaSuccess ||
            cudaMalloc((void **)&h->ring_flags, (size_t)(2 * depth + 1) * 32 * sizeof(int)) != cudaSuccess) {
            (void)cudaGetLastError();
            return PLSPEC_ERR_ALLOC;
        }
        PL_CUDA(h, cudaMemsetAsync(h->ring_flags + 64 * depth, 0, sizeof(int), stream));   // error word (see finalize)
        h->ring_depth = depth; h->ring_ctas = cta_max;
    }
    long long vg = (long long)g_cnt * Q;
    const int n_cta = vg < cta_max ? (int)vg : cta_max;   // a multiple of Q either way
    const int GR = n_cta / Q, rounds = (g_cnt + GR - 1) / GR;
    // producer inputs through shared memory if two buffers + the slice's twiddles fit beside the exchange regions
    // (same arithmetic as the kernel: plspec_fused.cuh, ring mode)
    const long long vesz = h->dtype == PLSPEC_SC16 ? 4 : 8;
    const long long npmax = (h->Nk / 2 + n_cta - 1) / n_cta;
    const long long rcp = 2 * npmax + 2, rvb = (((long long)(GR - 1) * h->stride + 2 * npmax) * vesz + 31) & ~15LL;
    const long long stage_bytes = 2 * Q * (rcp * 8 + rvb) + (long long)(Q - 1) * 2 * npmax * 8;
    const int staged = h->opt_stage && stage_bytes <= (long long)kStageMaxBytes ? 1 : 0;
    const size_t smem = (size_t)kStageOff + (staged ? (size_t)stage_bytes : 0);
    int per_launch = (1 << 20) / rounds;                  // IPPs per launch: counters stay far below 2^31
    if (per_launch < 1) return PLSPEC_ERR_UNSUPPORTED;
    const size_t esz = h->dtype == PLSPEC_SC16 ? 4 : 8;
    const int c_pitch = h->opt_shared_code ? 0 : h->L;
    for (int p0 = 0; p0 < n_ipp; p0 += per_launch) {
        const int nb = n_ipp - p0 < per_launch ? n_ipp - p0 : per_launch;
        PL_CUDA(h, cudaMemsetAsync(h->ring_flags, 0, (size_t)2 * depth * 32 * sizeof(int), stream));
        KParams P{};
        P.V = (const char *)dV + (size_t)p0 * (size_t)v_pitch * esz;
        P.C = dC + (size_t)p0 * (size_t)c_pitch;
        P.S = h->S + (size_t)g_lo * (size_t)h->N; P.twA = h->twA; P.twB = h->twB; P.twN = h->twN;
        P.Cbits = nullptr; P.not_bpsk = nullptr; P.epoch = 1;
        P.v_pitch = v_pitch;
        P.N = h->N; P.Nk = h->Nk; P.Q = Q; P.log2Nk = ilog2(h->Nk);
        P.L = h->L; P.R = g_cnt; P.r0 = r0 + g_lo * h->stride; P.stride = h->stride;
        P.n_groups = rounds; P.n_ipp = nb; P.n_chunks = 0; P.use_atomic = 1;
        P.ring = h->ring; P.ring_flags = h->ring_flags; P.ring_depth = depth; P.ring_ahead = ahead; P.c_pitch = c_pitch;
        P.ring_stage = staged;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)n_cta);
        cfg.blockDim = dim3(kFusedThreads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeCooperative;      // the CTAs wait on one another: all must be resident
        attr[0].val.cooperative = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        void *args[] = {&P};
        PL_CUDA(h, cudaLaunchKernelExC(&cfg, h->kfunc_ring, args));
        h->stats.kernel_launches++;
        h->stats.ipp_chunks_last = 0;
    }
    return PLSPEC_OK;
}

// N > 16384, PLSPEC_OPT_SPLIT = 1 (default): predecode_kernel (every window decoded once, outer radix-Q butterfly) -> scratch -> fused
// kernel with Q = 1 over g_cnt * Q virtual gates, in batches of IPPs that fit the scratch buffer.
int launch_split(plspec_ctx *h, const void *dV, const float2 *dC, long long v_pitch, int r0, int n_ipp, int g_lo,
                 int g_cnt, cudaStream_t stream) {
    const long long per_ipp_full = (long long)h->R * h->N;             // float2 elements of scratch per IPP, all gates
    const long long per_ipp = (long long)g_cnt * h->N;                 // ... of this launch's gates
    if (!h->xq) {
        long long want = (4LL << 30) / (per_ipp_full * (long long)sizeof(float2));   // <= 4 GiB
        if (want < 1) want = 1;
        if (want > 64) want = 64;
        if (h->opt_batch > 0 && want > h->opt_batch) want = h->opt_batch;
        while (want >= 1 && cudaMalloc((void **)&h->xq, (size_t)(want * per_ipp_full) * sizeof(float2)) != cudaSuccess) {
            (void)cudaGetLastError();
            h->xq = nullptr;
            want /= 2;
        }
        if (!h->xq) return PLSPEC_ERR_ALLOC;
        h->xq_ipps = want;
    }
    long long fit = h->xq_ipps * per_ipp_full / per_ipp;               // IPPs of g_cnt gates the scratch holds
    if (h->opt_batch > 0 && fit > h->opt_batch) fit = h->opt_batch;
    if (fit > 65535) fit = 65535;
    const size_t esz = h->dtype == PLSPEC_SC16 ? 4 : 8;
    for (int p0 = 0; p0 < n_ipp; p0 += (int)fit) {
        const int nb = n_ipp - p0 < (int)fit ? n_ipp - p0 : (int)fit;
        KParams P{};
        P.V = (const char *)dV + (size_t)p0 * (size_t)v_pitch * esz;
        const int c_pitch = h->opt_shared_code ? 0 : h->L;            // the pre-pass reads the one code in place
        P.C = dC + (size_t)p0 * (size_t)c_pitch;
        P.S = h->S + (size_t)g_lo * (size_t)h->N; P.twA = h->twA; P.twB = h->twB; P.twN = h->twN;
        P.Cbits = nullptr; P.not_bpsk = nullptr; P.epoch = 1;
        P.v_pitch = v_pitch;
        P.N = h->N; P.Nk = h->Nk; P.Q = h->Q; P.log2Nk = ilog2(h->Nk);
        P.L = h->L; P.R = g_cnt; P.r0 = r0 + g_lo * h->stride; P.stride = h->stride;
        P.n_groups = g_cnt; P.n_ipp = nb; P.n_chunks = 1; P.use_atomic = 0;
        P.ring = nullptr; P.ring_flags = nullptr; P.ring_depth = 0; P.ring_ahead = 0; P.c_pitch = c_pitch; P.ring_stage = 0;
        constexpr int GB = 8;                                         // gates per thread of the pre-pass
        if ((g_cnt + GB - 1) / GB > 65535) return PLSPEC_ERR_UNSUPPORTED;
        const dim3 blocks((unsigned)(h->Nk / 512), (unsigned)((g_cnt + GB - 1) / GB), (unsigned)nb);
        const bool sc = h->dtype == PLSPEC_SC16;
        if (h->Q == 2) {
            if (sc) predecode_kernel<2, DT_SC16, GB><<<blocks, 256, 0, stream>>>(P, h->xq);
            else    predecode_kernel<2, DT_CF32, GB><<<blocks, 256, 0, stream>>>(P, h->xq);
        } else {
            if (sc) predecode_kernel<4, DT_SC16, GB><<<blocks, 256, 0, stream>>>(P, h->xq);
            else    predecode_kernel<4, DT_CF32, GB><<<blocks, 256, 0, stream>>>(P, h->xq);
        }
        PL_CUDA(h, cudaGetLastError());
        h->stats.kernel_launches++;
        // step 2: g_cnt * Q virtual gates, window = Nk contiguous decoded samples, identity code
        KParams F = P;
        F.V = h->xq; F.C = dC;
        F.Cbits = nullptr; F.not_bpsk = nullptr; F.epoch = 1;         // the kernel variant takes the windows as decoded
        F.v_pitch = per_ipp;
        F.N = h->Nk; F.Q = 1; F.L = h->Nk;
        F.R = g_cnt * h->Q; F.r0 = 0; F.stride = h->Nk;
        F.n_groups = F.R;
        const long long items = (long long)F.n_groups * nb;
        long long tiles;
        if (h->opt_chunks > 0) {
            F.n_chunks = h->opt_chunks < nb ? h->opt_chunks : nb;
            tiles = (long long)F.n_groups * F.n_chunks;
        } else {
            F.n_chunks = 0;
            tiles = items < h->slots_per_wave ? items : h->slots_per_wave;
        }
        F.use_atomic = 1;
        h->stats.ipp_chunks_last = F.n_chunks;
        if (tiles > 0x7fffffffLL) return PLSPEC_ERR_UNSUPPORTED;
        void *args[] = {&F};
        PL_CUDA(h, launch_fused(h->kfunc_split, (unsigned)tiles, (unsigned)kFusedThreads, args, (size_t)kStageOff, stream,
                                true));
        h->stats.kernel_launches++;
    }
    return PLSPEC_OK;
}

// order this call's work after everything accumulated before on another stream
int chain_streams(plspec_ctx *h, cudaStream_t stream) {
    if (h->have_work && h->last_stream != stream) PL_CUDA(h, cudaStreamWaitEvent(stream, h->work_done, 0));
    return PLSPEC_OK;
}
int mark_work(plspec_ctx *h, cudaStream_t stream) {
    PL_CUDA(h, cudaEventRecord(h->work_done, stream));
    h->last_stream = stream;
    h->have_work = true;
    return PLSPEC_OK;
}

int ensure_slots(plspec_ctx *h, int batch) {
    if (h->slot_batch >= batch) return PLSPEC_OK;
    const size_t esz = h->dtype == PLSPEC_SC16 ? 4 : 8;
    for (int s = 0; s < kSlots; s++) {
        Slot &sl = h->slot[s];
        if (sl.used) PL_CUDA(h, cudaEventSynchronize(sl.freed));
        if (sl.V) cudaFree(sl.V);
        if (sl.C) cudaFree(sl.C);
        sl.V = nullptr; sl.C = nullptr; sl.used = false;
        if (cudaMalloc(&sl.V, (size_t)batch * h->span * esz) != cudaSuccess ||
            cudaMalloc((void **)&sl.C, (size_t)batch * h->L * sizeof(float2)) != cudaSuccess) {
            (void)cudaGetLastError();
            h->slot_batch = 0;
            return PLSPEC_ERR_ALLOC;
        }
        if (!sl.ready) PL_CUDA(h, cudaEventCreateWithFlags(&sl.ready, cudaEventDisableTiming));
        if (!sl.freed) PL_CUDA(h, cudaEventCreateWithFlags(&sl.freed, cudaEventDisableTiming));
    }
    h->slot_batch = batch;
    return PLSPEC_OK;
}

// copy the needed span of IPPs [p0, p0 + nb) of a host-buffer call, and their codes, on the copy stream
int copy_ipps(plspec_ctx *h, const void *V, const void *C, int p0, int nb, void *dV, float2 *dC) {
    const size_t esz = h->dtype == PLSPEC_SC16 ? 4 : 8;
    const char *src = (const char *)V + ((size_t)p0 * h->ipp_len + h->r0) * esz;
    PL_CUDA(h, cudaMemcpy2DAsync(dV, (size_t)h->span * esz, src, (size_t)h->ipp_len * esz, (size_t)h->span * esz, nb,
                                 cudaMemcpyHostToDevice, h->copy_stream));
    const size_t c_off = h->opt_shared_code ? 0 : (size_t)p0 * h->L * sizeof(float2);
    const size_t c_bytes = (size_t)(h->opt_shared_code ? 1 : nb) * h->L * sizeof(float2);
    PL_CUDA(h, cudaMemcpyAsync(dC, (const char *)C + c_off, c_bytes, cudaMemcpyHostToDevice, h->copy_stream));
    h->stats.h2d_bytes += (long long)nb * (long long)h->span * (long long)esz + (long long)c_bytes;
    return PLSPEC_OK;
}

// The deferred IPPs (struct Tail) are transformed now, over all gates, on `stream`.
int flush_tail(plspec_ctx *h, cudaStream_t stream) {
    Tail &t = h->tail;
    if (!t.pending) return PLSPEC_OK;
    t.pending = false;
    const int rc = launch_gates(h, t.cp, t.V, h->span, 0, t.n_ipp, 0, h->R, stream);   // codes prepared when they were copied
    if (rc != PLSPEC_OK) return rc;
    PL_CUDA(h, cudaEventRecord(t.done, stream));
    t.used = true;
    return PLSPEC_OK;
}

// Host-resident inputs: copy only the needed span of each IPP (PAPER.md:149 item 3) in batches
// on the copy stream, overlapped with the kernels of earlier batches (PAPER.md:149 item 2).
int accumulate_from_host(plspec_ctx *h, const void *V, const void *C, int n_ipp, cudaStream_t stream) {
    const size_t esz = h->dtype == PLSPEC_SC16 ? 4 : 8;
    const size_t per_ipp = (size_t)h->span * esz + (h->opt_shared_code ? 0 : (size_t)h->L * sizeof(float2));
    // the last part of the call's IPPs (as far as they fit kTailMaxBytes) is staged but left for plspec_finalize
    // (or the next plspec_accumulate): see struct Tail
    // How many: half, or more where the write-out is long against the transform (large N, few pulses): the deferred
    // transform should last ~1.3x the device -> host copy of S that hides under it.  Estimates: 5 N log2 N flop per
    // window at half the FP32 peak; 50 GB/s for the copy.
    double frac = 0.5;
    {
        const double t_d2h = (double)h->R * h->N * 4.0 / 50e9;
        const double t_all = (double)n_ipp * h->R * 5.0 * h->N * (double)ilog2(h->N) / 37e12;
        const double want = 1.3 * t_d2h / (t_all > 0 ? t_all : 1.0);
        frac = want < 0.5 ? 0.5 : (want > 0.75 ? 0.75 : want);
    }
    int n_tail = h->opt_defer ? (int)(n_ipp * frac + 0.999) : 0;
    if (n_tail > n_ipp) n_tail = n_ipp;
    const size_t tail_cap = kTailMaxBytes / per_ipp;
    if ((size_t)n_tail > tail_cap) n_tail = (int)tail_cap;
    const int n_head = n_ipp - n_tail;
    int rc;
    if (n_head > 0) {
        // auto: eight batches per call, but none below ~4 MB (each batch pays the launches' fixed cost once)
        int batch = (n_head + 7) / 8;
        const int min_batch = (int)(((size_t)4 << 20) / per_ipp) + 1;
        if (batch < min_batch) batch = min_batch;
        if (h->opt_batch > 0) batch = h->opt_batch;
        const int cap = (int)((256u << 20) / per_ipp);        // <= 256 MiB per slot
        if (batch > cap) batch = cap;
        if (batch < 1) batch = 1;
        if (batch > n_head) batch = n_head;
        if ((rc = ensure_slots(h, batch)) != PLSPEC_OK) return rc;
        for (int p0 = 0; p0 < n_head; p0 += batch) {
            const int nb = n_head - p0 < batch ? n_head - p0 : batch;
            Slot &sl = h->slot[h->next_slot];
            h->next_slot = (h->next_slot + 1) % kSlots;
            if (sl.used) PL_CUDA(h, cudaStreamWaitEvent(h->copy_stream, sl.freed, 0));
            if ((rc = copy_ipps(h, V, C, p0, nb, sl.V, sl.C)) != PLSPEC_OK) return rc;
            PL_CUDA(h, cudaEventRecord(sl.ready, h->copy_stream));
            PL_CUDA(h, cudaStreamWaitEvent(stream, sl.ready, 0));
            rc = launch_accumulate(h, sl.V, sl.C, h->span, 0, nb, stream);
            if (rc) return rc;
            PL_CUDA(h, cudaEventRecord(sl.freed, stream));
            sl.used = true;
        }
    }
    if (n_tail > 0) {
        Tail &t = h->tail;
        const size_t v_need = (size_t)n_tail * h->span * esz;
        const size_t c_need = (size_t)(h->opt_shared_code ? 1 : n_tail) * h->L * sizeof(float2);
        if (t.used) PL_CUDA(h, cudaStreamWaitEvent(h->copy_stream, t.done, 0));   // kernels of the previous tail
        if (v_need > t.v_bytes || c_need > t.c_bytes) {
            if (t.V) cudaFree(t.V);                                // cudaFree waits for the device
            if (t.C) cudaFree(t.C);
            t.V = nullptr; t.C = nullptr; t.v_bytes = t.c_bytes = 0;
            if (cudaMalloc(&t.V, v_need) != cudaSuccess || cudaMalloc((void **)&t.C, c_need) != cudaSuccess) {
                (void)cudaGetLastError();
                return PLSPEC_ERR_ALLOC;
            }
            t.v_bytes = v_need; t.c_bytes = c_need;
        }
        if (!t.ready) PL_CUDA(h, cudaEventCreateWithFlags(&t.ready, cudaEventDisableTiming));
        if (!t.done) PL_CUDA(h, cudaEventCreateWithFlags(&t.done, cudaEventDisableTiming));
        if ((rc = copy_ipps(h, V, C, n_head, n_tail, t.V, t.C)) != PLSPEC_OK) return rc;
        PL_CUDA(h, cudaEventRecord(t.ready, h->copy_stream));
        PL_CUDA(h, cudaStreamWaitEvent(stream, t.ready, 0));
        t.cp.flag = 2;
        if ((rc = prepare_codes(h, t.cp, t.C, n_tail, stream)) != PLSPEC_OK) return rc;   // with the options of this call
        t.n_ipp = n_tail;
        t.pending = true;
    }
    return PLSPEC_OK;
}

int build_tables(plspec_ctx *h) {
    // full circle W_N^e, correctly rounded from float64 (never a recurrence)
    std::vector<float2> t((size_t)h->N);
    for (int e = 0; e < h->N; e++) {
        double a = -2.0 * M_PI * (double)e / (double)h->N;
        t[e] = make_float2((float)cos(a), (float)sin(a));
    }
    PL_CUDA(h, cudaMalloc((void **)&h->twN, sizeof(float2) * (size_t)h->N));
    PL_CUDA(h, cudaMemcpy(h->twN, t.data(), sizeof(float2) * (size_t)h->N, cudaMemcpyHostToDevice));
    // fused kernel tables (plspec_fused.cuh), every entry rounded once from float64
    const int Nk = h->N < kMaxNk ? h->N : kMaxNk;
    if (Nk >= 1024) {
        const int RA = Nk / 1024;
        // pass A -> B1: W_Nk^{t_lo f_hi}, t_lo = 64 a' + lane + 32 o, packed over o: [a'][f_hi][re/im][lane]
        std::vector<float2> u((size_t)Nk);
        for (int ap = 0; ap < 16; ap++)
            for (int f = 0; f < RA; f++)
                for (int lane = 0; lane < 32; lane++) {
                    double w[2][2];
                    for (int o = 0; o < 2; o++) {
                        const long long t_lo = 64 * ap + lane + 32 * o;
                        const double a = -2.0 * M_PI * (double)((t_lo * f) % Nk) / (double)Nk;
                        w[o][0] = cos(a); w[o][1] = sin(a);
                    }
                    for (int k = 0; k < 2; k++)
                        u[(size_t)((ap * RA + f) * 2 + k) * 32 + lane] = make_float2((float)w[0][k], (float)w[1][k]);
                }
        PL_CUDA(h, cudaMalloc((void **)&h->twA, sizeof(float2) * (size_t)Nk));
        PL_CUDA(h, cudaMemcpy(h->twA, u.data(), sizeof(float2) * (size_t)Nk, cudaMemcpyHostToDevice));
        // pass B1 -> B2: W_1024^{b c}, packed over (c', c' + 16): [c'][re/im][b]
        std::vector<float2> v(1024);
        for (int c = 0; c < 16; c++)
            for (int b = 0; b < 32; b++) {
                const double a0 = -2.0 * M_PI * (double)((b * c) % 1024) / 1024.0;
                const double a1 = -2.0 * M_PI * (double)((b * (c + 16)) % 1024) / 1024.0;
                v[(size_t)(c * 2 + 0) * 32 + b] = make_float2((float)cos(a0), (float)cos(a1));
                v[(size_t)(c * 2 + 1) * 32 + b] = make_float2((float)sin(a0), (float)sin(a1));
            }
        PL_CUDA(h, cudaMalloc((void **)&h->twB, sizeof(float2) * 1024));
        PL_CUDA(h, cudaMemcpy(h->twB, v.data(), sizeof(float2) * 1024, cudaMemcpyHostToDevice));
    }
    return PLSPEC_OK;
}

void free_ctx(plspec_ctx *h) {
    if (!h) return;
    (void)cudaDeviceSynchronize();
    for (int s = 0; s < kSlots; s++) {
        if (h->slot[s].V) cudaFree(h->slot[s].V);
        if (h->slot[s].C) cudaFree(h->slot[s].C);
        if (h->slot[s].ready) cudaEventDestroy(h->slot[s].ready);
        if (h->slot[s].freed) cudaEventDestroy(h->slot[s].freed);
    }
    if (h->S) cudaFree(h->S);
    if (h->S_tmp) cudaFree(h->S_tmp);
    if (h->prod_work) cudaFree(h->prod_work);
    if (h->twA) cudaFree(h->twA);
    if (h->twB) cudaFree(h->twB);
    if (h->twN) cudaFree(h->twN);
    for (CodePrep *cp : {&h->cp, &h->tail.cp}) {
        if (cp->cbits) cudaFree(cp->cbits);
        if (cp->crep) cudaFree(cp->crep);
    }
    if (h->tail.V) cudaFree(h->tail.V);
    if (h->tail.C) cudaFree(h->tail.C);
    if (h->tail.ready) cudaEventDestroy(h->tail.ready);
    if (h->tail.done) cudaEventDestroy(h->tail.done);
    if (h->d2h_stream) cudaStreamDestroy(h->d2h_stream);
    for (int k = 0; k < kMaxRanges; k++)
        if (h->range_done[k]) cudaEventDestroy(h->range_done[k]);
    if (h->xq) cudaFree(h->xq);
    if (h->ring) cudaFree(h->ring);
    if (h->ring_flags) cudaFree(h->ring_flags);
    if (h->not_bpsk) cudaFree(h->not_bpsk);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    if (h->work_done) cudaEventDestroy(h->work_done);
    (void)cudaGetLastError();
    delete h;
}

// 1 = device-accessible (device / managed), 0 = host (pinned or pageable), <0 error
int pointer_is_device(plspec_ctx *h, const void *p, int *is_dev) {
    cudaPointerAttributes a;
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { (void)cudaGetLastError(); h->last_cuda = (int)e; return PLSPEC_ERR_CUDA; }
    *is_dev = (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) ? 1 : 0;
    return PLSPEC_OK;
}

}  // namespace

extern "C" {

int plspec_create(int N, int code_len, int n_ranges, int r0, int stride, int ipp_len, int dtype,
                  plspec_handle *out) {
    if (!out) return PLSPEC_ERR_INVALID_ARG;
    *out = nullptr;
    if (!is_pow2(N) || N < 16 || N > 65536) return PLSPEC_ERR_INVALID_ARG;
    if (code_len < 1 || code_len > N || n_ranges < 1 || r0 < 0 || stride < 1 || ipp_len < 0)
        return PLSPEC_ERR_INVALID_ARG;
    if (dtype != PLSPEC_CF32 && dtype != PLSPEC_SC16) return PLSPEC_ERR_INVALID_ARG;
    const long long span = (long long)(n_ranges - 1) * stride + code_len;
    if (span + r0 > 0x7fffffffLL) return PLSPEC_ERR_INVALID_ARG;
    if (ipp_len == 0) ipp_len = (int)(span + r0);
    if (span + r0 > ipp_len) return PLSPEC_ERR_INVALID_ARG;

    plspec_ctx *h = new (std::nothrow) plspec_ctx();
    if (!h) return PLSPEC_ERR_ALLOC;
    memset(&h->stats, 0, sizeof(h->stats));
    h->N = N; h->L = code_len; h->R = n_ranges; h->r0 = r0; h->stride = stride;
    h->ipp_len = ipp_len; h->dtype = dtype; h->span = (int)span;

    int rc = PLSPEC_OK;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDevice(&h->device);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, h->device);
    if (e != cudaSuccess) { (void)cudaGetLastError(); delete h; return PLSPEC_ERR_CUDA; }
    if (prop.major != 10 || prop.minor != 0) { delete h; return PLSPEC_ERR_UNSUPPORTED; }   // the library holds sm_100a code only
    h->n_sm = prop.multiProcessorCount;

    auto fail = [&](int code) { free_ctx(h); return code; };
    const size_t s_bytes = sizeof(float) * (size_t)n_ranges * (size_t)N;
    if (cudaMalloc((void **)&h->S, s_bytes) != cudaSuccess) { (void)cudaGetLastError(); return fail(PLSPEC_ERR_ALLOC); }
    if (cudaMemset(h->S, 0, s_bytes) != cudaSuccess) { (void)cudaGetLastError(); return fail(PLSPEC_ERR_CUDA); }
    if (cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&h->d2h_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->work_done, cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(PLSPEC_ERR_CUDA);
    }
    for (int k = 0; k < kMaxRanges; k++)
        if (cudaEventCreateWithFlags(&h->range_done[k], cudaEventDisableTiming) != cudaSuccess) {
            (void)cudaGetLastError();
            return fail(PLSPEC_ERR_CUDA);
        }
    if (cudaMalloc((void **)&h->not_bpsk, 4 * sizeof(int)) != cudaSuccess) { (void)cudaGetLastError(); return fail(PLSPEC_ERR_ALLOC); }
    if (cudaMemset(h->not_bpsk, 0, 4 * sizeof(int)) != cudaSuccess) { (void)cudaGetLastError(); return fail(PLSPEC_ERR_CUDA); }
    if ((rc = build_tables(h)) != PLSPEC_OK) return fail(rc);
    if ((rc = select_kernel(h)) != PLSPEC_OK) return fail(rc);
    *out = h;
    return PLSPEC_OK;
}

int plspec_configure(plspec_handle h, int option, int value) {
    if (!h || value < 0) return PLSPEC_ERR_INVALID_ARG;
    switch (option) {
        case PLSPEC_OPT_KERNEL: {
            if (value > 2) return PLSPEC_ERR_INVALID_ARG;
            if (h->have_work) return PLSPEC_ERR_INVALID_ARG;   // the two kernels lay S_dev out differently
            const int old = h->opt_kernel;
            h->opt_kernel = value;
            int rc = select_kernel(h);
            if (rc != PLSPEC_OK) { h->opt_kernel = old; (void)select_kernel(h); }
            return rc;
        }
        case PLSPEC_OPT_IPP_CHUNKS: h->opt_chunks = value; return PLSPEC_OK;
        case PLSPEC_OPT_H2D_BATCH:  h->opt_batch = value;  return PLSPEC_OK;
        case PLSPEC_OPT_BPSK_PACK:  if (value > 1) return PLSPEC_ERR_INVALID_ARG; h->opt_bpsk = value; return PLSPEC_OK;
        case PLSPEC_OPT_SHARED_CODE:
            if (value > 1) return PLSPEC_ERR_INVALID_ARG;
            h->opt_shared_code = value;
            return PLSPEC_OK;
        case PLSPEC_OPT_DEFER:
            if (value > 1) return PLSPEC_ERR_INVALID_ARG;
            h->opt_defer = value;
            return PLSPEC_OK;
        case PLSPEC_OPT_RING_DEPTH:
            if (value < 2 || value > 16) return PLSPEC_ERR_INVALID_ARG;
            h->opt_ring_depth = value;
            if (h->opt_ring_ahead >= value) h->opt_ring_ahead = value - 1;
            return PLSPEC_OK;
        case PLSPEC_OPT_RING_AHEAD:
            if (value < 1 || value >= h->opt_ring_depth) return PLSPEC_ERR_INVALID_ARG;
            h->opt_ring_ahead = value;
            return PLSPEC_OK;
        case PLSPEC_OPT_SPLIT: {
            if (value > 2) return PLSPEC_ERR_INVALID_ARG;
            if (h->have_work) return PLSPEC_ERR_INVALID_ARG;
            h->opt_split = value;
            return select_kernel(h);
        }
        case PLSPEC_OPT_STAGE: {
            if (value > 2) return PLSPEC_ERR_INVALID_ARG;
            const int old = h->opt_stage;
            h->opt_stage = value;
            int rc = select_kernel(h);
            if (rc != PLSPEC_OK) { h->opt_stage = old; (void)select_kernel(h); }
            return rc;
        }
    }
    return PLSPEC_ERR_INVALID_ARG;
}

int plspec_accumulate(plspec_handle h, const void *voltages, const void *codes, int n_ipp, void *stream_) {
    if (!h || n_ipp < 0) return PLSPEC_ERR_INVALID_ARG;
    if (n_ipp == 0) return PLSPEC_OK;
    if (!voltages || !codes) return PLSPEC_ERR_INVALID_ARG;
    cudaStream_t stream = (cudaStream_t)stream_;
    int vdev = 0, cdev = 0, rc;
    if ((rc = pointer_is_device(h, voltages, &vdev)) != PLSPEC_OK) return rc;
    if ((rc = pointer_is_device(h, codes, &cdev)) != PLSPEC_OK) return rc;
    if (vdev != cdev) return PLSPEC_ERR_INVALID_ARG;
    if ((rc = chain_streams(h, stream)) != PLSPEC_OK) return rc;
    if ((rc = flush_tail(h, stream)) != PLSPEC_OK) return rc;        // deferred IPPs of the previous call come first
    if (vdev) rc = launch_accumulate(h, voltages, (const float2 *)codes, h->ipp_len, h->r0, n_ipp, stream);
    else      rc = accumulate_from_host(h, voltages, codes, n_ipp, stream);
    if (rc != PLSPEC_OK) return rc;
    h->stats.ipps_accumulated += n_ipp;
    return mark_work(h, stream);
}

int plspec_finalize(plspec_handle h, float *S_out) {
    if (!h || !S_out) return PLSPEC_ERR_INVALID_ARG;
    int out_dev = 0, rc;
    if ((rc = pointer_is_device(h, S_out, &out_dev)) != PLSPEC_OK) return rc;
    cudaStream_t st = h->last_stream;
    const size_t total = (size_t)h->R * (size_t)h->N;
    const bool permuted = h->Q > 1 || h->kind == 2;       // S_dev is not in natural bin order
    if (out_dev && (rc = flush_tail(h, st)) != PLSPEC_OK) return rc;
    if (!out_dev && !h->S_tmp && cudaMalloc((void **)&h->S_tmp, total * sizeof(float)) != cudaSuccess) {
        (void)cudaGetLastError();
        return PLSPEC_ERR_ALLOC;
    }
    // Gate ranges.  Device S_out: one.  Host S_out: up to kMaxRanges of >= ~8 MB; range k is transformed (the deferred
    // IPPs, if any), un-permuted into S_tmp and copied out on the d2h stream while range k + 1 computes.  Equal ranges
    // keep the copy stream and the kernels in step (where the copy of S takes about as long as the deferred transform,
    // cfg 4, a small first range leaves the copy stream waiting for the large second one); only the last range is
    // smaller (S / 16, within 2 ... 8 MB): its copy is the part nothing overlaps.
    const int n_groups = (h->R + h->gates_per_cta - 1) / h->gates_per_cta;
    int n_ranges = 1;
    int bound[kMaxRanges + 1];                            // gate groups: range k = [bound[k], bound[k + 1])
    bound[0] = 0;
    if (!out_dev) {
        const double s_bytes = (double)total * sizeof(float), mb = (double)(1 << 20);
        const size_t want = (size_t)(s_bytes / (8 * mb));
        n_ranges = want < 1 ? 1 : (want > (size_t)kMaxRanges ? kMaxRanges : (int)want);
        if (n_ranges > n_groups) n_ranges = n_groups;
        double last = 1.0 / n_ranges;                     // fraction of the gates in the last range
        if (n_ranges >= 4) {
            double edge = s_bytes / 16;
            edge = edge < 2 * mb ? 2 * mb : (edge > 8 * mb ? 8 * mb : edge);
            if (edge / s_bytes < last) last = edge / s_bytes;
        }
        for (int k = 1; k < n_ranges; k++) bound[k] = (int)((1.0 - last) * n_groups * k / (n_ranges - 1) + 0.5);
        for (int k = 1; k < n_ranges; k++)                // strictly increasing, inside (0, n_groups)
            if (bound[k] <= bound[k - 1] || bound[k] >= n_groups) { n_ranges = 1; break; }
    }
    bound[n_ranges] = n_groups;
    Tail &t = h->tail;
    const bool tail = t.pending;
    t.pending = false;
    const int RAe = h->kind == 2 ? h->RA : 1, NC = h->kind == 2 ? 1024 : h->Nk, M = h->Q * RAe;
    const int TC = 4096 / M < NC ? 4096 / M : NC;
    for (int k = 0; k < n_ranges; k++) {
        const int g_lo = bound[k] * h->gates_per_cta;
        int g_hi = bound[k + 1] * h->gates_per_cta;
        if (g_hi > h->R) g_hi = h->R;
        const int g_cnt = g_hi - g_lo;
        const size_t off = (size_t)g_lo * (size_t)h->N, cnt = (size_t)g_cnt * (size_t)h->N;
        if (tail && (rc = launch_gates(h, t.cp, t.V, h->span, 0, t.n_ipp, g_lo, g_cnt, st)) != PLSPEC_OK) return rc;
        float *dst = (out_dev ? S_out : h->S_tmp) + off;
        if (permuted) {
            // one pass: transposition to natural bin order + zeroing of the accumulators
            finalize_kernel<<<dim3((unsigned)g_cnt, (unsigned)(NC / TC)), 256, (size_t)TC * (M + 1) * sizeof(float), st>>>(
                h->S + off, dst, ilog2(h->Q), ilog2(RAe), NC, TC);
            PL_CUDA(h, cudaGetLastError());
            h->stats.kernel_launches++;
        } else {
            PL_CUDA(h, cudaMemcpyAsync(dst, h->S + off, cnt * sizeof(float), cudaMemcpyDeviceToDevice, st));
            PL_CUDA(h, cudaMemsetAsync(h->S + off, 0, cnt * sizeof(float), st));
        }
        if (!out_dev) {
            PL_CUDA(h, cudaEventRecord(h->range_done[k], st));
            PL_CUDA(h, cudaStreamWaitEvent(h->d2h_stream, h->range_done[k], 0));
            PL_CUDA(h, cudaMemcpyAsync(S_out + off, dst, cnt * sizeof(float), cudaMemcpyDeviceToHost, h->d2h_stream));
            h->stats.d2h_bytes += (long long)(cnt * sizeof(float));
        }
    }
    if (tail) {
        PL_CUDA(h, cudaEventRecord(t.done, st));
        t.used = true;
    }
    PL_CUDA(h, cudaStreamSynchronize(st));
    if (!out_dev) PL_CUDA(h, cudaStreamSynchronize(h->d2h_stream));
    h->have_work = false;
    if (h->ring_flags) {                                  // a ring-mode wait gave up: the spectra are not to be trusted
        int err = 0;
        PL_CUDA(h, cudaMemcpy(&err, h->ring_flags + 64 * h->ring_depth, sizeof(int), cudaMemcpyDeviceToHost));
        if (err) {
            (void)cudaMemset(h->ring_flags + 64 * h->ring_depth, 0, sizeof(int));
            h->last_cuda = (int)cudaErrorLaunchTimeout;
            return PLSPEC_ERR_CUDA;
        }
    }
    return PLSPEC_OK;
}

int plspec_finalize_products(plspec_handle h, float *S_out, const plspec_products_t *prod) {
    if (!h || !S_out || !prod) return PLSPEC_ERR_INVALID_ARG;
    const bool want_prof = prod->k_up || prod->p_up || prod->k_dn || prod->p_dn || prod->noise;
    if (want_prof && !(prod->k_up && prod->p_up && prod->k_dn && prod->p_dn && prod->noise)) return PLSPEC_ERR_INVALID_ARG;
    if (prod->n_ipp < 1 || (prod->centred != 0 && prod->centred != 1)) return PLSPEC_ERR_INVALID_ARG;
    if (want_prof && (prod->k_min < 1 || prod->k_min >= h->N / 2 || prod->guard < 0)) return PLSPEC_ERR_INVALID_ARG;
    if (prod->P_out == S_out) return PLSPEC_ERR_INVALID_ARG;
    const void *ptrs[] = {S_out, prod->P_out, prod->k_up, prod->p_up, prod->k_dn, prod->p_dn, prod->noise};
    for (const void *p : ptrs) {                         // device (or managed) memory only
        if (!p) continue;
        int dev = 0, rc = pointer_is_device(h, p, &dev);
        if (rc != PLSPEC_OK) return rc;
        if (!dev) return PLSPEC_ERR_INVALID_ARG;
    }
    if (((uintptr_t)S_out & 15) || ((uintptr_t)prod->P_out & 15)) return PLSPEC_ERR_INVALID_ARG;
    cudaStream_t st = h->last_stream;
    int rc = flush_tail(h, st);
    if (rc != PLSPEC_OK) return rc;
    const size_t total = (size_t)h->R * (size_t)h->N;
    if (h->Q > 1 || h->kind == 2) {
        // one pass over S_dev: transposition to natural order, zeroing, mean spectrum and line search
        const int RAe = h->kind == 2 ? h->RA : 1, NC = h->kind == 2 ? 1024 : h->Nk, M = h->Q * RAe;
        const int TC = 4096 / M < NC ? 4096 / M : NC;
        ProductsWork *work = nullptr;
        if (want_prof) {
            if (!h->prod_work && cudaMalloc((void **)&h->prod_work, sizeof(ProductsWork) * (size_t)h->R) != cudaSuccess) {
                (void)cudaGetLastError();
                return PLSPEC_ERR_ALLOC;
            }
            work = static_cast<ProductsWork *>(h->prod_work);
            PL_CUDA(h, cudaMemsetAsync(work, 0, sizeof(ProductsWork) * (size_t)h->R, st));
        }
        finalize_products_kernel<<<dim3((unsigned)h->R, (unsigned)(NC / TC)), 256, (size_t)TC * (M + 1) * sizeof(float), st>>>(
            h->S, S_out, ilog2(h->Q), ilog2(RAe), NC, TC, prod->P_out, prod->centred, prod->n_ipp, prod->k_min, work);
        PL_CUDA(h, cudaGetLastError());
        h->stats.kernel_launches++;
        if (want_prof) {
            products_tail_kernel<<<(unsigned)((h->R + 3) / 4), 128, 0, st>>>(S_out, work, h->R, h->N, prod->n_ipp, prod->k_min,
                                                                            prod->guard, prod->k_up, prod->p_up, prod->k_dn,
                                                                            prod->p_dn, prod->noise);
            PL_CUDA(h, cudaGetLastError());
            h->stats.kernel_launches++;
        }
    } else {
        // generic kernel, N <= 16384: S_dev is in natural order already; the stand-alone product kernels follow the copy
        PL_CUDA(h, cudaMemcpyAsync(S_out, h->S, total * sizeof(float), cudaMemcpyDeviceToDevice, st));
        PL_CUDA(h, cudaMemsetAsync(h->S, 0, total * sizeof(float), st));
        if (prod->P_out && (rc = plspec_mean_spectrum(S_out, prod->P_out, h->R, h->N, prod->n_ipp, prod->centred, st)) != PLSPEC_OK)
            return rc;
        if (want_prof && (rc = plspec_profile(S_out, h->R, h->N, prod->n_ipp, prod->k_min, prod->guard, prod->k_up, prod->p_up,
                                              prod->k_dn, prod->p_dn, prod->noise, st)) != PLSPEC_OK)
            return rc;
        h->stats.kernel_launches += (prod->P_out ? 1 : 0) + (want_prof ? 1 : 0);
    }
    PL_CUDA(h, cudaStreamSynchronize(st));
    h->have_work = false;
    return PLSPEC_OK;
}

int plspec_profile(const float *S, int n_ranges, int N, int n_ipp, int k_min, int guard, int *k_up, float *p_up,
                   int *k_dn, float *p_dn, float *noise, void *stream) {
    if (!S || !k_up || !p_up || !k_dn || !p_dn || !noise) return PLSPEC_ERR_INVALID_ARG;
    if (!is_pow2(N) || N < 16 || N > 65536 || n_ranges < 1 || n_ipp < 1 || k_min < 1 || k_min >= N / 2 || guard < 0)
        return PLSPEC_ERR_INVALID_ARG;
    const void *ptrs[] = {S, k_up, p_up, k_dn, p_dn, noise};
    for (const void *p : ptrs) {                         // device (or managed) memory only
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return PLSPEC_ERR_CUDA; }
        if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged) return PLSPEC_ERR_INVALID_ARG;
    }
    if ((uintptr_t)S & 15) return PLSPEC_ERR_INVALID_ARG;  // rows are read in 128-bit loads
    profile_kernel<<<(unsigned)n_ranges, kProfileThreads, 0, (cudaStream_t)stream>>>(S, N, n_ipp, k_min, guard, k_up, p_up, k_dn,
                                                                         p_dn, noise);
    if (cudaGetLastError() != cudaSuccess) return PLSPEC_ERR_CUDA;
    return PLSPEC_OK;
}

int plspec_mean_spectrum(const float *S, float *P_out, int n_ranges, int N, int n_ipp, int centred, void *stream) {
    if (!S || !P_out || S == P_out) return PLSPEC_ERR_INVALID_ARG;
    if (!is_pow2(N) || N < 16 || N > 65536 || n_ranges < 1 || n_ipp < 1 || (centred != 0 && centred != 1))
        return PLSPEC_ERR_INVALID_ARG;
    const void *ptrs[] = {S, P_out};
    for (const void *p : ptrs) {                         // device (or managed) memory only, 16-byte aligned
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return PLSPEC_ERR_CUDA; }
        if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged) return PLSPEC_ERR_INVALID_ARG;
        if ((uintptr_t)p & 15) return PLSPEC_ERR_INVALID_ARG;
    }
    const long long n_vec = (long long)n_ranges * (N / 4);
    long long blocks = (n_vec + 255) / 256;
    const int n_sm = device_sm_count();
    if (n_sm < 1) return PLSPEC_ERR_CUDA;
    if (blocks > n_sm * 8) blocks = n_sm * 8;            // grid-stride: eight CTAs of 256 per SM
    mean_spectrum_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>((const float4 *)S, (float4 *)P_out, n_vec,
                                                                             ilog2(N), n_ipp, centred);
    if (cudaGetLastError() != cudaSuccess) return PLSPEC_ERR_CUDA;
    return PLSPEC_OK;
}

int plspec_diag_fp32_peak(int packed, int iters, int reps, double *tflops_best, double *tflops_mean, void *stream_) {
    if ((packed != 0 && packed != 1) || iters < 1 || reps < 1 || reps > 100000 || !tflops_best || !tflops_mean)
        return PLSPEC_ERR_INVALID_ARG;
    cudaStream_t stream = (cudaStream_t)stream_;
    const int n_sm = device_sm_count();
    if (n_sm < 1) return PLSPEC_ERR_CUDA;
    const unsigned grid = (unsigned)n_sm * 4, block = 512;            // 2048 resident threads per SM
    float *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = PLSPEC_OK;
    if (cudaMalloc((void **)&sink, sizeof(float)) != cudaSuccess) { (void)cudaGetLastError(); return PLSPEC_ERR_ALLOC; }
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = PLSPEC_ERR_CUDA;
    const double flop = (double)grid * block * (double)iters * 64.0;  // 32 multiply-adds per thread and iteration
    double best = 0.0, sum = 0.0;
    for (int r = -1; r < reps && rc == PLSPEC_OK; r++) {              // r = -1: warm-up launch, not counted
        cudaEventRecord(e0, stream);
        if (packed) fma_peak_kernel<true><<<grid, block, 0, stream>>>(sink, 0.999f, 0.001f, iters);
        else        fma_peak_kernel<false><<<grid, block, 0, stream>>>(sink, 0.999f, 0.001f, iters);
        cudaEventRecord(e1, stream);
        float ms = 0.f;
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess || ms <= 0.f) {
            rc = PLSPEC_ERR_CUDA;
            break;
        }
        if (r < 0) continue;
        const double tf = flop / ((double)ms * 1e-3) / 1e12;
        if (tf > best) best = tf;
        sum += tf;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    if (rc != PLSPEC_OK) { (void)cudaGetLastError(); return rc; }
    *tflops_best = best;
    *tflops_mean = sum / reps;
    return PLSPEC_OK;
}

int plspec_diag_mem_bandwidth(int kind, long long bytes, int n_ctas, int passes, double *gbs, void *stream_) {
    if (kind < 0 || kind > 3 || bytes < (1 << 20) || bytes > (8LL << 30) || n_ctas < 1 || n_ctas > 65535 || passes < 1 || !gbs)
        return PLSPEC_ERR_INVALID_ARG;
    cudaStream_t stream = (cudaStream_t)stream_;
    bytes &= ~((long long)(1 << 20) - 1);                              // whole MiB
    if (kind == 3 && bytes / n_ctas < 16384) return PLSPEC_ERR_INVALID_ARG;   // a CTA's share: at least one bulk store
    unsigned char *buf = nullptr;
    uint4 *sink = nullptr;
    if (cudaMalloc((void **)&buf, (size_t)bytes) != cudaSuccess || cudaMalloc((void **)&sink, sizeof(uint4)) != cudaSuccess) {
        (void)cudaGetLastError();
        if (buf) cudaFree(buf);
        return PLSPEC_ERR_ALLOC;
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = PLSPEC_OK;
    if (cudaMemsetAsync(buf, 0, (size_t)bytes, stream) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
        cudaEventCreate(&e1) != cudaSuccess)
        rc = PLSPEC_ERR_CUDA;
    const size_t nvec = (size_t)bytes / 16;
    double moved = (double)bytes * passes;                             // bytes read + written by one launch
    if (kind == 3) moved = (double)(((size_t)bytes / n_ctas) & ~(size_t)16383) * n_ctas * passes;
    double best_ms = 0.0;
    for (int r = -1; r < 3 && rc == PLSPEC_OK; r++) {                  // r = -1: warm-up (also brings the buffer into L2)
        cudaEventRecord(e0, stream);
        switch (kind) {
            case 0: bw_read_kernel<<<n_ctas, 512, 0, stream>>>((const uint4 *)buf, nvec, passes, sink); break;
            case 1: bw_write_kernel<<<n_ctas, 512, 0, stream>>>((uint4 *)buf, nvec, passes); break;
            case 2: bw_copy_kernel<<<n_ctas, 512, 0, stream>>>((uint4 *)buf, nvec, passes); break;
            default: bw_tma_store_kernel<<<n_ctas, 512, 0, stream>>>(buf, (size_t)bytes, passes); break;
        }
        cudaEventRecord(e1, stream);
        float ms = 0.f;
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess || ms <= 0.f) {
            rc = PLSPEC_ERR_CUDA;
            break;
        }
        if (r >= 0 && (best_ms == 0.0 || ms < best_ms)) best_ms = ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    cudaFree(sink);
    if (rc != PLSPEC_OK) { (void)cudaGetLastError(); return rc; }
    *gbs = moved / (best_ms * 1e-3) / 1e9;
    return PLSPEC_OK;
}

int plspec_reset(plspec_handle h) {
    if (!h) return PLSPEC_ERR_INVALID_ARG;
    cudaStream_t st = h->last_stream;
    h->tail.pending = false;                              // deferred IPPs are dropped with the rest
    PL_CUDA(h, cudaMemsetAsync(h->S, 0, sizeof(float) * (size_t)h->R * (size_t)h->N, st));
    PL_CUDA(h, cudaStreamSynchronize(st));
    h->have_work = false;
    return PLSPEC_OK;
}

int plspec_destroy(plspec_handle h) {
    free_ctx(h);
    return PLSPEC_OK;
}

int plspec_get_stats(plspec_handle h, plspec_stats_t *out) {
    if (!h || !out) return PLSPEC_ERR_INVALID_ARG;
    *out = h->stats;
    return PLSPEC_OK;
}

int plspec_last_cuda_error(plspec_handle h) { return h ? h->last_cuda : 0; }

const char *plspec_strerror(int status) {
    switch (status) {
        case PLSPEC_OK: return "ok";
        case PLSPEC_ERR_INVALID_ARG: return "invalid argument";
        case PLSPEC_ERR_ALLOC: return "allocation failed";
        case PLSPEC_ERR_CUDA: return "CUDA call failed (see plspec_last_cuda_error)";
        case PLSPEC_ERR_UNSUPPORTED: return "unsupported on this device or build";
    }
    return "unknown status";
}

const char *plspec_version(void) { return "plspec 0.1 (sm_100a)"; }

}  // extern "C"
