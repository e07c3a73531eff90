// beagle.cu — libbeagle_b200.so: the C-ABI of include/beagle.h and every kernel behind it.
//
// Hot path:
//   a2  k_block_sums / k_scan_block_sums            exclusive prefix sum of lengths -> off[]
//   a3  k_program_scan / k_bins_and_cases / k_scatter
//                                                    per-program scan (max stack depth, well-formedness),
//                                                    counting sort by (depth class, length) -> perm[]
//   a4  k_bins_and_cases + TMA in the eval kernel   X,y transposed/padded once, bulk-copied per CTA
//   a5-a7  k_eval_* (eval_kernel.inc)               fetch, decode, interpret, reduce, tax, store
//   a8  beagle_eval_chunked                         double-buffered H2D on a copy stream
// PyTorch is not involved: only the CUDA runtime. sm_100a only.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/beagle.h"
#include "ops.cuh"

namespace beagle {

// ---- opcode numbers on the device side (include/beagle.h) -------------------------------------------
enum : uint32_t { UOP_END = 0, OPC_CONST = BEAGLE_OP_CONST, OPC_LOAD = BEAGLE_OP_LOAD, OPC_ADD = BEAGLE_OP_ADD,
                  OPC_SUB = BEAGLE_OP_SUB, OPC_MUL = BEAGLE_OP_MUL, OPC_DIV = BEAGLE_OP_DIV,
                  OPC_SIN = BEAGLE_OP_SIN, OPC_COS = BEAGLE_OP_COS, OPC_LOG = BEAGLE_OP_LOG,
                  OPC_SQRT = BEAGLE_OP_SQRT, OPC_EXP = BEAGLE_OP_EXP, UOP_MOV0 = 12 };

constexpr int kNumClasses = 3;                 // depth classes: <=8, <=16, <=32 stack entries
constexpr int kClassDepth[kNumClasses] = { 8, 16, 32 };
constexpr int kNumBins = BEAGLE_MAX_LEN + 1;   // bin = 512 - length  (longest first)
constexpr int kScanThreads = 256;              // programs per block in the pre-pass
constexpr int kEvalThreads = 384;              // 12 warps: 65536 regs / 384 = 170 per thread
constexpr int kUopBytes = (BEAGLE_MAX_LEN + 4) * 8;
constexpr int kRawBytes = (BEAGLE_MAX_LEN + 8) * 4;
constexpr int kWarpBytes = 2 * kUopBytes + 2 * kRawBytes;
constexpr int kProfMax = 256;                  // beagle_set_profiling: recorded calls
constexpr int kCasePad = 512;                  // staged cases are padded to a multiple of 32*K for every K

struct Header {                                // device-resident results of the pre-pass
    long long T;                               // total tokens = sum of in-range lengths
    int cls_start[kNumClasses + 1];            // perm[] range of each depth class
    unsigned int queue[kNumClasses];           // work-queue cursors of the evaluation kernels
    int n_malformed;
};

struct EvalParams {
    const int32_t* genomes; const long long* off; const int32_t* lengths; const int32_t* perm;
    const float* consts; const float* xt; const Header* hdr; unsigned int* queue;
    float* fitness; float* outputs;
    float tax; int n; int npad; int d; int cls;
};

// ---- PTX helpers: mbarrier, TMA bulk copy, cp.async --------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n"
        ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void tma_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cp_async_16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_4(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ int clamp_len(int l) { return (l >= 1 && l <= BEAGLE_MAX_LEN) ? l : 0; }

// ---- a2: offsets ------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kScanThreads) k_block_sums(const int32_t* __restrict__ lengths, long long P,
                                                             long long* __restrict__ bsum)
{
    __shared__ int wsum[kScanThreads / 32];
    const long long p = (long long)blockIdx.x * kScanThreads + threadIdx.x;
    int v = (p < P) ? clamp_len(lengths[p]) : 0;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) t += wsum[w];
        bsum[blockIdx.x] = t;
    }
}

// one block: exclusive scan of the block sums in place; also clears the bins and the header
__global__ void __launch_bounds__(1024) k_scan_block_sums(long long* __restrict__ bsum, int nblocks,
                                                          Header* __restrict__ hdr, int* __restrict__ bins)
{
    __shared__ long long wtot[32];
    __shared__ long long carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    for (int i = threadIdx.x; i < 2 * kNumClasses * kNumBins; i += blockDim.x) bins[i] = 0;  // counts + cursors
    __syncthreads();
    for (int base = 0; base < nblocks; base += 1024) {
        const int i = base + threadIdx.x;
        long long v = (i < nblocks) ? bsum[i] : 0, inc = v;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) { long long o = __shfl_up_sync(0xffffffffu, inc, s); if (lane >= s) inc += o; }
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            long long w = wtot[lane], winc = w;
#pragma unroll
            for (int s = 1; s < 32; s <<= 1) { long long o = __shfl_up_sync(0xffffffffu, winc, s); if (lane >= s) winc += o; }
            wtot[lane] = winc - w;
        }
        __syncthreads();
        const long long carry = carry_s;
        if (i < nblocks) bsum[i] = carry + wtot[warp] + inc - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = carry + wtot[31] + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        hdr->T = carry_s;
        hdr->n_malformed = 0;
        for (int c = 0; c < kNumClasses; ++c) hdr->queue[c] = 0;
    }
}

// ---- a3: per-program scan, histogram of (depth class, length) ------------------------------------------
// One thread per program: off[p], then one walk over its tokens (max stack depth, well-formedness:
// DESIGN.md D3). Malformed individuals get the canonical NaN here and never reach the interpreter.
__global__ void __launch_bounds__(kScanThreads) k_program_scan(
    const int32_t* __restrict__ genomes, const int32_t* __restrict__ lengths, long long P,
    const long long* __restrict__ bsum, long long n_consts, int d,
    long long* __restrict__ off, int* __restrict__ key, int* __restrict__ depth_out,
    int* __restrict__ bins, float* __restrict__ fitness, float* __restrict__ outputs, int n_cases,
    Header* __restrict__ hdr)
{
    __shared__ int wsum[kScanThreads / 32];
    __shared__ int hist[kNumClasses * kNumBins];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kNumClasses * kNumBins; i += kScanThreads) hist[i] = 0;
    const long long p = (long long)blockIdx.x * kScanThreads + threadIdx.x;
    const int raw_len = (p < P) ? lengths[p] : 0;
    const int len = clamp_len(raw_len);
    int inc = len;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, s); if (lane >= s) inc += o; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    int wbase = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) wbase += (w < warp) ? wsum[w] : 0;
    const long long o = bsum[blockIdx.x] + wbase + inc - len;
    if (p < P) {
        off[p] = o;
        int sp = 0, mx = 0;
        bool ok = len > 0;
        const uint32_t* tok = reinterpret_cast<const uint32_t*>(genomes) + o;
        for (int t = 0; t < len; ++t) {
            const uint32_t w = __ldg(tok + t);
            const uint32_t op = tok_op(w), arg = tok_arg(w);
            if (op == OPC_CONST) { ok &= ((long long)arg < n_consts); ++sp; }
            else if (op == OPC_LOAD) { ok &= ((int)arg < d); ++sp; }
            else if (op >= OPC_ADD && op <= OPC_DIV) { ok &= (arg == 0) & (sp >= 2); --sp; }
            else if (op >= OPC_SIN && op <= OPC_EXP) { ok &= (arg == 0) & (sp >= 1); }
            else ok = false;
            ok &= (sp <= BEAGLE_MAX_STACK);
            mx = max(mx, sp);
            if (!ok) break;
        }
        ok &= (sp >= 1);
        int k = -1;
        if (ok) {
            const int cls = mx <= kClassDepth[0] ? 0 : (mx <= kClassDepth[1] ? 1 : 2);
            k = cls * kNumBins + (BEAGLE_MAX_LEN - len);
            atomicAdd(&hist[k], 1);
        } else {
            if (fitness) fitness[p] = __uint_as_float(0x7FC00000u);
            if (outputs) for (int i = 0; i < n_cases; ++i) outputs[(size_t)p * n_cases + i] = __uint_as_float(0x7FC00000u);
            atomicAdd(&hdr->n_malformed, 1);
        }
        key[p] = k;
        depth_out[p] = ok ? mx : 0;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kNumClasses * kNumBins; i += kScanThreads)
        if (hist[i]) atomicAdd(&bins[i], hist[i]);
}

// one block: exclusive scan of the bins -> bin starts and class ranges; and a4's transpose of the
// fitness cases into the variable-major, zero-padded block every evaluation CTA bulk-copies.
__global__ void __launch_bounds__(1024) k_bins_and_cases(const int* __restrict__ bins, int* __restrict__ binstart,
                                                         Header* __restrict__ hdr,
                                                         const float* __restrict__ X, const float* __restrict__ y,
                                                         int n, int d, int npad, float* __restrict__ xt)
{
    __shared__ int wtot[32];
    __shared__ int carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    constexpr int total = kNumClasses * kNumBins;
    for (int base = 0; base < total; base += 1024) {
        const int i = base + threadIdx.x;
        int v = (i < total) ? bins[i] : 0, inc = v;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, s); if (lane >= s) inc += o; }
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            int w = wtot[lane], winc = w;
#pragma unroll
            for (int s = 1; s < 32; s <<= 1) { int o = __shfl_up_sync(0xffffffffu, winc, s); if (lane >= s) winc += o; }
            wtot[lane] = winc - w;
        }
        __syncthreads();
        const int carry = carry_s;
        const int ex = carry + wtot[warp] + inc - v;
        if (i < total) {
            binstart[i] = ex;
            if (i % kNumBins == 0) hdr->cls_start[i / kNumBins] = ex;
        }
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = carry + wtot[31] + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) hdr->cls_start[kNumClasses] = carry_s;
    // transpose: xt[j][i] = X[i][j] (j < d), xt[d][i] = y[i]; cases i >= n are zero
    for (int e = threadIdx.x; e < (d + 1) * npad; e += blockDim.x) {
        const int j = e / npad, i = e - j * npad;
        float v = 0.f;
        if (i < n) v = (j < d) ? X[(size_t)i * d + j] : (y ? y[i] : 0.f);
        xt[e] = v;
    }
}

__global__ void __launch_bounds__(kScanThreads) k_scatter(const int* __restrict__ key, long long P,
                                                          const int* __restrict__ binstart, int* __restrict__ cursor,
                                                          int* __restrict__ perm)
{
    __shared__ int cnt[kNumClasses * kNumBins];
    for (int i = threadIdx.x; i < kNumClasses * kNumBins; i += kScanThreads) cnt[i] = 0;
    __syncthreads();
    const long long p = (long long)blockIdx.x * kScanThreads + threadIdx.x;
    const int k = (p < P) ? key[p] : -1;
    int r = 0;
    if (k >= 0) r = atomicAdd(&cnt[k], 1);
    __syncthreads();
    // one global reservation per (block, non-empty bin); cnt[] becomes the block's base in that bin
    for (int i = threadIdx.x; i < kNumClasses * kNumBins; i += kScanThreads)
        if (cnt[i]) cnt[i] = atomicAdd(&cursor[i], cnt[i]);
    __syncthreads();
    if (k >= 0) perm[binstart[k] + cnt[k] + r] = (int)p;
}

// ---- the evaluation kernels: one instantiation per depth class ------------------------------------------
#define BG_NAME k_eval_k16d8
#define BG_K 16
#define BG_D 8
#define BG_SLOTS(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7)
#define BG_SLOTS_BIN(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6)
#include "eval_kernel.inc"
#undef BG_NAME
#undef BG_K
#undef BG_D
#undef BG_SLOTS
#undef BG_SLOTS_BIN

#define BG_NAME k_eval_k8d16
#define BG_K 8
#define BG_D 16
#define BG_SLOTS(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15)
#define BG_SLOTS_BIN(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14)
#include "eval_kernel.inc"
#undef BG_NAME
#undef BG_K
#undef BG_D
#undef BG_SLOTS
#undef BG_SLOTS_BIN

#define BG_NAME k_eval_k4d32
#define BG_K 4
#define BG_D 32
#define BG_SLOTS(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15) \
    M(16) M(17) M(18) M(19) M(20) M(21) M(22) M(23) M(24) M(25) M(26) M(27) M(28) M(29) M(30) M(31)
#define BG_SLOTS_BIN(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15) \
    M(16) M(17) M(18) M(19) M(20) M(21) M(22) M(23) M(24) M(25) M(26) M(27) M(28) M(29) M(30)
#include "eval_kernel.inc"
#undef BG_NAME
#undef BG_K
#undef BG_D
#undef BG_SLOTS
#undef BG_SLOTS_BIN

// ---- prior art as a baseline: the paper's mapping ------------------------------------------
// One block per individual, one thread per fitness case, a 32-entry per-thread stack in local
// memory, every thread decodes every token. The residuals go through shared memory so that warp 0
// can add them in the canonical order: results are bit-identical to the warp-per-individual kernels.
__global__ void __launch_bounds__(1024) k_eval_blockwise(
    const int32_t* __restrict__ genomes, const long long* __restrict__ off, const int32_t* __restrict__ lengths,
    const int* __restrict__ depth, const float* __restrict__ consts, const float* __restrict__ X,
    const float* __restrict__ y, int n, int d, float tax, float* __restrict__ fitness)
{
    __shared__ float res[BEAGLE_MAX_N];
    const int p = blockIdx.x;
    if (depth[p] == 0) return;                 // malformed: NaN already written by the pre-pass
    const int len = lengths[p];
    const uint32_t* tok = reinterpret_cast<const uint32_t*>(genomes) + off[p];
    const int i = threadIdx.x;
    if (i < n) {
        float st[BEAGLE_MAX_STACK];
        int sp = 0;
        for (int t = 0; t < len; ++t) {
            const uint32_t w = __ldg(tok + t);
            const uint32_t op = tok_op(w), arg = tok_arg(w);
            switch (op) {
            case OPC_CONST: st[sp++] = __ldg(consts + arg); break;
            case OPC_LOAD: st[sp++] = __ldg(X + (size_t)i * d + arg); break;
            case OPC_ADD: st[sp - 2] = op_add(st[sp - 2], st[sp - 1]); --sp; break;
            case OPC_SUB: st[sp - 2] = op_sub(st[sp - 2], st[sp - 1]); --sp; break;
            case OPC_MUL: st[sp - 2] = op_mul(st[sp - 2], st[sp - 1]); --sp; break;
            case OPC_DIV: st[sp - 2] = op_div(st[sp - 2], st[sp - 1]); --sp; break;
            case OPC_SIN: st[sp - 1] = op_sin(st[sp - 1]); break;
            case OPC_COS: st[sp - 1] = op_cos(st[sp - 1]); break;
            case OPC_LOG: st[sp - 1] = op_log(st[sp - 1]); break;
            case OPC_SQRT: st[sp - 1] = op_sqrt(st[sp - 1]); break;
            case OPC_EXP: st[sp - 1] = op_exp(st[sp - 1]); break;
            default: break;
            }
        }
        res[i] = __fsub_rn(st[sp - 1], __ldg(y + i));
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        float acc = 0.f;
        for (int m = 0; m * 128 < n; ++m)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int ci = m * 128 + lane * 4 + e;
                if (ci < n) { const float r = res[ci]; acc = __fmaf_rn(r, r, acc); }
            }
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) acc = __fadd_rn(acc, __shfl_xor_sync(0xffffffffu, acc, m));
        if (lane == 0) fitness[p] = __fmaf_rn(tax, (float)len, __fdiv_rn(acc, (float)n));
    }
}

// ======================================================================================================
//                                        host side
// ======================================================================================================
struct Workspace {
    long long cap_P = 0;
    long long* off = nullptr; int* key = nullptr; int* depth = nullptr; int* perm = nullptr;
    long long* bsum = nullptr; int* bins = nullptr; int* binstart = nullptr; float* xt = nullptr;
    Header* hdr = nullptr;
    // chunked staging
    long long stage_bytes = 0; unsigned char* stage[2] = { nullptr, nullptr };
    float* stage_consts = nullptr; long long stage_consts_cap = 0;
    cudaStream_t copy_stream = nullptr; cudaEvent_t ev_copied[2] = { nullptr, nullptr }, ev_free[2] = { nullptr, nullptr };
    cudaEvent_t ev_k[2 * kProfMax] = {}; int prof_n = 0;
    int num_sms = 0; int smem_optin = 0; bool device_ok = false; bool inited = false;
};
static Workspace g_ws;
static int32_t g_last_cuda = 0;
static int32_t g_launches = 0;
static int32_t g_profiling = 0;

#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { g_last_cuda = (int32_t)e_; \
    return (e_ == cudaErrorMemoryAllocation) ? BEAGLE_ERR_NOMEM : BEAGLE_ERR_CUDA; } } while (0)

static beagle_status init_once()
{
    Workspace& w = g_ws;
    if (w.inited) return w.device_ok ? BEAGLE_OK : BEAGLE_ERR_UNSUPPORTED;
    int dev = 0; CU(cudaGetDevice(&dev));
    cudaDeviceProp prop; CU(cudaGetDeviceProperties(&prop, dev));
    w.num_sms = prop.multiProcessorCount;
    w.smem_optin = (int)prop.sharedMemPerBlockOptin;
    w.device_ok = (prop.major == 10);
    w.inited = true;
    if (!w.device_ok) return BEAGLE_ERR_UNSUPPORTED;
    CU(cudaFuncSetAttribute(k_eval_k16d8, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval_k8d16, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval_k4d32, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaMalloc(&w.bins, sizeof(int) * 2 * kNumClasses * kNumBins));
    CU(cudaMalloc(&w.binstart, sizeof(int) * kNumClasses * kNumBins));
    CU(cudaMalloc(&w.xt, sizeof(float) * (BEAGLE_MAX_D + 1) * BEAGLE_MAX_N));
    CU(cudaMalloc(&w.hdr, sizeof(Header)));
    return BEAGLE_OK;
}

static beagle_status reserve_P(long long P)
{
    Workspace& w = g_ws;
    if (P <= w.cap_P) return BEAGLE_OK;
    CU(cudaDeviceSynchronize());
    cudaFree(w.off); cudaFree(w.key); cudaFree(w.depth); cudaFree(w.perm); cudaFree(w.bsum);
    w.off = nullptr; w.key = nullptr; w.depth = nullptr; w.perm = nullptr; w.bsum = nullptr; w.cap_P = 0;
    const long long nb = (P + kScanThreads - 1) / kScanThreads;
    CU(cudaMalloc(&w.off, sizeof(long long) * (P + 1)));
    CU(cudaMalloc(&w.key, sizeof(int) * P));
    CU(cudaMalloc(&w.depth, sizeof(int) * P));
    CU(cudaMalloc(&w.perm, sizeof(int) * P));
    CU(cudaMalloc(&w.bsum, sizeof(long long) * (nb + 1)));
    w.cap_P = P;
    return BEAGLE_OK;
}

static beagle_status check_args(const void* genomes, const void* lengths, int64_t P, const void* consts,
                                int64_t n_consts, const void* X, const void* y, int32_t N, int32_t d, const void* out)
{
    if (P < 0 || P > 0x7FFFFFFFll) return BEAGLE_ERR_INVALID_ARG;
    if (N < 1 || N > BEAGLE_MAX_N || d < 1 || d > BEAGLE_MAX_D) return BEAGLE_ERR_INVALID_ARG;
    if (n_consts < 0 || n_consts > BEAGLE_MAX_CONSTS) return BEAGLE_ERR_INVALID_ARG;
    if (n_consts > 0 && !consts) return BEAGLE_ERR_INVALID_ARG;
    if (P > 0 && (!genomes || !lengths || !X || !y || !out)) return BEAGLE_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(genomes) & 3) || (reinterpret_cast<uintptr_t>(lengths) & 3)) return BEAGLE_ERR_INVALID_ARG;
    return BEAGLE_OK;
}

// a2 + a3 (+ the transpose of a4). After this: off, depth, perm, hdr are valid on `st`.
static beagle_status run_prepass(const int32_t* genomes, const int32_t* lengths, long long P, long long n_consts,
                                 const float* X, const float* y, int N, int d, float* fitness, float* outputs,
                                 cudaStream_t st)
{
    Workspace& w = g_ws;
    const int nb = (int)((P + kScanThreads - 1) / kScanThreads);
    const int npad = (N + kCasePad - 1) / kCasePad * kCasePad;
    k_block_sums<<<nb, kScanThreads, 0, st>>>(lengths, P, w.bsum);
    k_scan_block_sums<<<1, 1024, 0, st>>>(w.bsum, nb, w.hdr, w.bins);
    k_program_scan<<<nb, kScanThreads, 0, st>>>(genomes, lengths, P, w.bsum, n_consts, d, w.off, w.key, w.depth,
                                                w.bins, fitness, outputs, N, w.hdr);
    k_bins_and_cases<<<1, 1024, 0, st>>>(w.bins, w.binstart, w.hdr, X, y, N, d, npad, w.xt);
    k_scatter<<<nb, kScanThreads, 0, st>>>(w.key, P, w.binstart, w.bins + kNumClasses * kNumBins, w.perm);
    g_launches += 5;
    CU(cudaGetLastError());
    return BEAGLE_OK;
}

static beagle_status run_eval(const int32_t* genomes, const int32_t* lengths, const float* consts, int N, int d,
                              float tax, float* fitness, float* outputs, cudaStream_t st)
{
    Workspace& w = g_ws;
    const int npad = (N + kCasePad - 1) / kCasePad * kCasePad;
    const long long xs_bytes = (long long)(d + 1) * npad * 4;
    const long long fixed = 128 + ((xs_bytes + 127) & ~127ll);
    int warps = (int)((w.smem_optin - fixed) / kWarpBytes);
    if (warps > kEvalThreads / 32) warps = kEvalThreads / 32;
    if (warps < 1) return BEAGLE_ERR_UNSUPPORTED;
    const size_t smem = (size_t)(fixed + (long long)warps * kWarpBytes);
    EvalParams prm;
    prm.genomes = genomes; prm.off = w.off; prm.lengths = lengths; prm.perm = w.perm; prm.consts = consts;
    prm.xt = w.xt; prm.hdr = w.hdr; prm.fitness = fitness; prm.outputs = outputs;
    prm.tax = tax; prm.n = N; prm.npad = npad; prm.d = d;
    const bool prof = g_profiling && w.prof_n < kProfMax;
    if (prof) {
        for (int i = 0; i < 2; ++i)
            if (!w.ev_k[2 * w.prof_n + i]) CU(cudaEventCreate(&w.ev_k[2 * w.prof_n + i]));
        CU(cudaEventRecord(w.ev_k[2 * w.prof_n], st));
    }
    for (int c = 0; c < kNumClasses; ++c) {
        prm.cls = c; prm.queue = &w.hdr->queue[c];
        if (c == 0) k_eval_k16d8<<<w.num_sms, warps * 32, smem, st>>>(prm);
        else if (c == 1) k_eval_k8d16<<<w.num_sms, warps * 32, smem, st>>>(prm);
        else k_eval_k4d32<<<w.num_sms, warps * 32, smem, st>>>(prm);
        ++g_launches;
    }
    if (prof) { CU(cudaEventRecord(w.ev_k[2 * w.prof_n + 1], st)); ++w.prof_n; }
    CU(cudaGetLastError());
    return BEAGLE_OK;
}

} // namespace beagle

using namespace beagle;

extern "C" {

beagle_status beagle_eval(const int32_t* genomes, const int32_t* lengths, int64_t P,
                          const float* consts, int64_t n_consts, const float* X, const float* y,
                          int32_t N, int32_t d, float tax, float* fitness_out, void* stream)
{
    beagle_status s = check_args(genomes, lengths, P, consts, n_consts, X, y, N, d, fitness_out);
    if (s != BEAGLE_OK) return s;
    g_launches = 0;
    if (P == 0) return BEAGLE_OK;
    if ((s = init_once()) != BEAGLE_OK) return s;
    if ((s = reserve_P(P)) != BEAGLE_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    if ((s = run_prepass(genomes, lengths, P, n_consts, X, y, N, d, fitness_out, nullptr, st)) != BEAGLE_OK) return s;
    return run_eval(genomes, lengths, consts, N, d, tax, fitness_out, nullptr, st);
}

beagle_status beagle_debug_outputs(const int32_t* genomes, const int32_t* lengths, int64_t P,
                                   const float* consts, int64_t n_consts, const float* X, int32_t N, int32_t d,
                                   float* out_PxN, void* stream)
{
    beagle_status s = check_args(genomes, lengths, P, consts, n_consts, X, X, N, d, out_PxN);
    if (s != BEAGLE_OK) return s;
    g_launches = 0;
    if (P == 0) return BEAGLE_OK;
    if ((s = init_once()) != BEAGLE_OK) return s;
    if ((s = reserve_P(P)) != BEAGLE_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    // y is not used for outputs; X's first column stands in so that the staging kernel has a valid pointer
    if ((s = run_prepass(genomes, lengths, P, n_consts, X, nullptr, N, d, nullptr, out_PxN, st)) != BEAGLE_OK) return s;
    return run_eval(genomes, lengths, consts, N, d, 0.f, nullptr, out_PxN, st);
}

beagle_status beagle_eval_blockwise(const int32_t* genomes, const int32_t* lengths, int64_t P,
                                    const float* consts, int64_t n_consts, const float* X, const float* y,
                                    int32_t N, int32_t d, float tax, float* fitness_out, void* stream)
{
    beagle_status s = check_args(genomes, lengths, P, consts, n_consts, X, y, N, d, fitness_out);
    if (s != BEAGLE_OK) return s;
    g_launches = 0;
    if (P == 0) return BEAGLE_OK;
    if ((s = init_once()) != BEAGLE_OK) return s;
    if ((s = reserve_P(P)) != BEAGLE_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    if ((s = run_prepass(genomes, lengths, P, n_consts, X, y, N, d, fitness_out, nullptr, st)) != BEAGLE_OK) return s;
    const int threads = (N + 31) / 32 * 32;
    k_eval_blockwise<<<(unsigned)P, threads, 0, st>>>(genomes, g_ws.off, lengths, g_ws.depth, consts, X, y, N, d, tax, fitness_out);
    ++g_launches;
    CU(cudaGetLastError());
    return BEAGLE_OK;
}

beagle_status beagle_debug_schedule(int64_t P, int64_t* off, int32_t* depth, int32_t* perm, void* stream)
{
    if (P < 0 || P > g_ws.cap_P) return BEAGLE_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (off) CU(cudaMemcpyAsync(off, g_ws.off, sizeof(long long) * P, cudaMemcpyDeviceToDevice, st));
    if (depth) CU(cudaMemcpyAsync(depth, g_ws.depth, sizeof(int) * P, cudaMemcpyDeviceToDevice, st));
    if (perm) CU(cudaMemcpyAsync(perm, g_ws.perm, sizeof(int) * P, cudaMemcpyDeviceToDevice, st));
    return BEAGLE_OK;
}

beagle_status beagle_reserve_chunked(int64_t device_budget_bytes)
{
    Workspace& w = g_ws;
    beagle_status s = init_once();
    if (s != BEAGLE_OK) return s;
    const long long half = (device_budget_bytes / 2) & ~255ll;
    if (half < 4ll * (BEAGLE_MAX_LEN + 1)) return BEAGLE_ERR_INVALID_ARG;
    if (!w.copy_stream) {
        CU(cudaStreamCreateWithFlags(&w.copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&w.ev_copied[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&w.ev_free[i], cudaEventDisableTiming));
        }
    }
    if (half != w.stage_bytes) {
        CU(cudaDeviceSynchronize());
        cudaFree(w.stage[0]); cudaFree(w.stage[1]); w.stage[0] = w.stage[1] = nullptr; w.stage_bytes = 0;
        CU(cudaMalloc(&w.stage[0], half));
        CU(cudaMalloc(&w.stage[1], half));
        w.stage_bytes = half;
    }
    return BEAGLE_OK;
}

beagle_status beagle_eval_chunked(const int32_t* h_genomes, const int32_t* h_lengths, int64_t P,
                                  const float* h_consts, int64_t n_consts, const float* X, const float* y,
                                  int32_t N, int32_t d, float tax, float* fitness_out,
                                  int64_t device_budget_bytes, void* stream)
{
    beagle_status s = check_args(h_genomes, h_lengths, P, h_consts, n_consts, X, y, N, d, fitness_out);
    if (s != BEAGLE_OK) return s;
    if (device_budget_bytes < 2ll * 4 * (BEAGLE_MAX_LEN + 1)) return BEAGLE_ERR_INVALID_ARG;
    g_launches = 0;
    if (P == 0) return BEAGLE_OK;
    if ((s = beagle_reserve_chunked(device_budget_bytes)) != BEAGLE_OK) return s;
    Workspace& w = g_ws;
    cudaStream_t st = (cudaStream_t)stream;
    // constants: copied whole, once (R19)
    if (n_consts > w.stage_consts_cap) {
        CU(cudaDeviceSynchronize());
        cudaFree(w.stage_consts); w.stage_consts = nullptr; w.stage_consts_cap = 0;
        CU(cudaMalloc(&w.stage_consts, sizeof(float) * n_consts));
        w.stage_consts_cap = n_consts;
    }
    // the copy stream must not start before work already queued on `stream` (e.g. the producer of X)
    CU(cudaEventRecord(w.ev_free[0], st)); CU(cudaStreamWaitEvent(w.copy_stream, w.ev_free[0], 0));
    CU(cudaEventRecord(w.ev_free[1], st));
    if (n_consts > 0)
        CU(cudaMemcpyAsync(w.stage_consts, h_consts, sizeof(float) * n_consts, cudaMemcpyHostToDevice, w.copy_stream));
    // chunk plan at individual boundaries: lengths first, then (16-byte aligned) tokens, in one staging
    // buffer: 4*(individuals + 3 + tokens) <= stage_bytes. The host scan that finds the end of chunk
    // c+1 runs while chunk c is being copied and evaluated.
    const long long cap_words = w.stage_bytes / 4 - 3;
    if ((s = reserve_P(P < cap_words ? P : cap_words)) != BEAGLE_OK) return s;
    long long p0 = 0, tok0 = 0;
    int total_launches = 0;
    for (int c = 0; p0 < P; ++c) {
        long long words = 0, p1 = p0, ntok = 0;
        while (p1 < P) {
            const int l = (h_lengths[p1] >= 1 && h_lengths[p1] <= BEAGLE_MAX_LEN) ? h_lengths[p1] : 0;
            if (words + l + 1 > cap_words) break;
            words += l + 1; ntok += l; ++p1;
        }
        const long long np = p1 - p0;
        const int b = c & 1;
        int32_t* d_len = reinterpret_cast<int32_t*>(w.stage[b]);
        int32_t* d_tok = d_len + ((np + 3) & ~3ll);
        CU(cudaStreamWaitEvent(w.copy_stream, w.ev_free[b], 0));      // buffer b is free again
        CU(cudaMemcpyAsync(d_len, h_lengths + p0, sizeof(int32_t) * np, cudaMemcpyHostToDevice, w.copy_stream));
        if (ntok > 0)
            CU(cudaMemcpyAsync(d_tok, h_genomes + tok0, sizeof(int32_t) * ntok, cudaMemcpyHostToDevice, w.copy_stream));
        CU(cudaEventRecord(w.ev_copied[b], w.copy_stream));
        CU(cudaStreamWaitEvent(st, w.ev_copied[b], 0));
        if ((s = run_prepass(d_tok, d_len, np, n_consts, X, y, N, d, fitness_out + p0, nullptr, st)) != BEAGLE_OK) return s;
        if ((s = run_eval(d_tok, d_len, w.stage_consts, N, d, tax, fitness_out + p0, nullptr, st)) != BEAGLE_OK) return s;
        CU(cudaEventRecord(w.ev_free[b], st));
        total_launches += g_launches; g_launches = 0;
        p0 = p1; tok0 += ntok;
    }
    g_launches = total_launches;
    return BEAGLE_OK;
}

void beagle_limits(int32_t* max_len, int32_t* max_stack, int32_t* max_n, int32_t* max_d)
{
    if (max_len) *max_len = BEAGLE_MAX_LEN;
    if (max_stack) *max_stack = BEAGLE_MAX_STACK;
    if (max_n) *max_n = BEAGLE_MAX_N;
    if (max_d) *max_d = BEAGLE_MAX_D;
}

const char* beagle_status_string(beagle_status s)
{
    switch (s) {
    case BEAGLE_OK: return "ok";
    case BEAGLE_ERR_INVALID_ARG: return "invalid argument";
    case BEAGLE_ERR_UNSUPPORTED: return "unsupported device or configuration (needs sm_100 and enough shared memory)";
    case BEAGLE_ERR_CUDA: return "CUDA error (see beagle_last_cuda_error)";
    case BEAGLE_ERR_NOMEM: return "out of device memory";
    default: return "unknown status";
    }
}

int32_t beagle_last_cuda_error(void) { return g_last_cuda; }

beagle_status beagle_reserve(int64_t P_max, int64_t T_max)
{
    (void)T_max;   // the workspace does not depend on the token count (tokens are read in place)
    if (P_max < 0 || P_max > 0x7FFFFFFFll) return BEAGLE_ERR_INVALID_ARG;
    beagle_status s = init_once();
    if (s != BEAGLE_OK) return s;
    return reserve_P(P_max);
}

void beagle_release(void)
{
    Workspace& w = g_ws;
    cudaDeviceSynchronize();
    cudaFree(w.off); cudaFree(w.key); cudaFree(w.depth); cudaFree(w.perm); cudaFree(w.bsum);
    cudaFree(w.stage[0]); cudaFree(w.stage[1]); cudaFree(w.stage_consts);
    w.off = nullptr; w.key = nullptr; w.depth = nullptr; w.perm = nullptr; w.bsum = nullptr; w.cap_P = 0;
    w.stage[0] = w.stage[1] = nullptr; w.stage_bytes = 0; w.stage_consts = nullptr; w.stage_consts_cap = 0;
}

int32_t beagle_last_launch_count(void) { return g_launches; }

void beagle_set_profiling(int32_t on) { g_profiling = on; if (on) g_ws.prof_n = 0; }

float beagle_profiled_eval_kernel_ms(int32_t* n_calls)
{
    Workspace& w = g_ws;
    if (n_calls) *n_calls = 0;
    if (w.prof_n <= 0) return -1.f;
    double sum = 0.0;
    for (int i = 0; i < w.prof_n; ++i) {
        float ms = 0.f;
        if (cudaEventSynchronize(w.ev_k[2 * i + 1]) != cudaSuccess) return -1.f;
        if (cudaEventElapsedTime(&ms, w.ev_k[2 * i], w.ev_k[2 * i + 1]) != cudaSuccess) return -1.f;
        sum += ms;
    }
    if (n_calls) *n_calls = w.prof_n;
    return (float)(sum / w.prof_n);
}

} // extern "C"
