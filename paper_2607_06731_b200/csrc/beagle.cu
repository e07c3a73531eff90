// beagle.cu — libbeagle_b200.so: the C-ABI of include/beagle.h and every kernel behind it.
//
// Hot path:
//   a2  k_len_pass1 / k_len_pass2      block sums + length histogram; exclusive scans -> offsets, bins
//   a3  k_scatter                      off[], counting sort by length (longest first) -> perm[]
//       k_compile                      per-program well-formedness, tree compile to micro-ops (uop.cuh):
//                                      terminal folding, fused fresh values, slot allocation
//   a4  k_len_pass2 + k_eval prologue  X,y transposed/padded once; X staged into tensor memory per CTA
//   a5-a7  k_eval (eval_kernel.inc)    TMA-fed interpreter: fetch, interpret, reduce, tax, store
//   a8  beagle_eval_chunked            double-buffered H2D on a copy stream
// PyTorch is not involved: only the CUDA runtime. sm_100a only.
// Test-only host builds of the device's integer logic (beagle_debug_prepass / _compile / _walk / _queue / _std_reward): the
// bodies of the pre-pass kernels, of the compiler's walk and of the interpreter's scheduling loop live in prepass_body.inc, walk_body.inc
// and queue_body.inc, included by the kernels with the device's macros and by host functions with plain C++ ones. No product path uses them.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <pthread.h>          // simt_host.inc (test only)
#include <map>
#include <atomic>
#include <mutex>
#include <system_error>
#include <string>
#include <thread>
#include <vector>

#include "../../include/beagle.h"
#include "ops.cuh"
#include "uop.cuh"
#include "interp.cuh"
#include "fit_corr.cuh"
#include "fit_std.cuh"
#include "rank.cuh"

namespace beagle {

// ---- opcode numbers on the device side (include/beagle.h) -------------------------------------------
enum : uint32_t { OPC_CONST = BEAGLE_OP_CONST, OPC_LOAD = BEAGLE_OP_LOAD, OPC_ADD = BEAGLE_OP_ADD,
                  OPC_SUB = BEAGLE_OP_SUB, OPC_MUL = BEAGLE_OP_MUL, OPC_DIV = BEAGLE_OP_DIV,
                  OPC_SIN = BEAGLE_OP_SIN, OPC_COS = BEAGLE_OP_COS, OPC_LOG = BEAGLE_OP_LOG,
                  OPC_SQRT = BEAGLE_OP_SQRT, OPC_EXP = BEAGLE_OP_EXP,
                  OPC_DUP = BEAGLE_OP_DUP, OPC_SWAP = BEAGLE_OP_SWAP, OPC_DEL = BEAGLE_OP_DEL,
                  OPC_SIGN = BEAGLE_OP_SIGN, OPC_SQUARE = BEAGLE_OP_SQUARE, OPC_CUBE = BEAGLE_OP_CUBE,
                  OPC_CBRT = BEAGLE_OP_CBRT, OPC_TAN = BEAGLE_OP_TAN, OPC_ARCSIN = BEAGLE_OP_ARCSIN,
                  OPC_ARCCOS = BEAGLE_OP_ARCCOS, OPC_ARCTAN = BEAGLE_OP_ARCTAN, OPC_TANH = BEAGLE_OP_TANH,
                  OPC_POW = BEAGLE_OP_POW, OPC_COPY = BEAGLE_OP_COPY, OPC_PASTE = BEAGLE_OP_PASTE };

constexpr int kNumBins = BEAGLE_MAX_LEN + 1;   // bin = 512 - length  (longest first); bin 512 unused
constexpr int kScanThreads = 256;              // threads per block in the pre-pass
constexpr int kScanItems = 8;                  // programs per thread: a block owns 2048 consecutive programs, so that the
                                               // per-(block, bin) global atomics are 8 times fewer
constexpr int kScanBlock = kScanThreads * kScanItems;
constexpr int kCompileThreads = 128;
constexpr int kStagesMax = 8;                  // micro-op stages in flight per warp
#ifndef BEAGLE_GROUP_STAGES
#define BEAGLE_GROUP_STAGES 2
#endif
#ifndef BEAGLE_GROUP_MAX
#define BEAGLE_GROUP_MAX 32
#endif
constexpr int kGroupMax = BEAGLE_GROUP_MAX;         // individuals per group at most (one visit to the queue brings 32)
constexpr int kGroupStages = BEAGLE_GROUP_STAGES;   // stages per ring when the longest program leaves room (eval_kernel.inc)
#ifndef BEAGLE_EVAL_THREADS
#define BEAGLE_EVAL_THREADS 1024
#endif
constexpr int kEvalThreads = BEAGLE_EVAL_THREADS;   // 32 warps (8 per scheduler): 64 registers per thread
constexpr int kStageBufsMax = 8;               // beagle_eval_chunked: staging buffers the device budget is cut into
constexpr long long kStageTarget = 32ll << 20;  // ... of about this size each (at least two); beagle_set_chunk_target overrides it
static long long g_stage_target = kStageTarget;
#ifndef BEAGLE_PLAN_W8
#define BEAGLE_PLAN_W8 0
#endif
constexpr int kProfMax = 256;                  // beagle_set_profiling: recorded calls
constexpr int kEvalMetaBytes = 64 * 16;           // per-warp window of the work queue (64 x int4)
constexpr int kCasePad = 512;                  // staged cases are padded to a multiple of 32*K
constexpr int kStageBytesMax = ((BEAGLE_MAX_LEN + 3 + 1) & ~1) * 8;   // 4128

struct Header {                                // device-resident results of the pre-pass
    long long T;                               // total tokens = sum of in-range lengths
    long long uop_entries;                     // micro-op entries reserved by the bins
    int n_sorted;                              // individuals with an in-range length (= entries of perm[])
    int max_len;                               // longest in-range length (>= 1 if n_sorted > 0)
    int n_slow;                                // individuals the blockwise kernel takes (POW, library functions, variables; or no room)
    int n_general;                             // individuals k_compile's walk turned down (k_compile_general)
    int n_f1;                                  // individuals compiled with DUP SWAP DEL SIGN SQUARE CUBE (picks k_compile<F1> next time)
    int n_malformed;
    unsigned int queue;                        // work-queue cursor of the interpreter kernel
    unsigned int queue2;                       // ... of the second launch of a split call
    unsigned int rcp_unsafe;                   // bit j: some case of variable j has |x| < 1e-6f (its division is protected)
};

struct EvalParams {
    const int4* meta; const uint2* uops; const Header* hdr; unsigned int* queue;
    const float* xt; const float* ung; float* fitness; float* outputs;
    float tax; float M; int power; int n; int npad; int d; int ring_bytes;   // M: the maximum score of the correlation fitness (f2)
    int rcp_col0;       // first tensor-memory column of the reciprocal rows: passes * d * 16
    int k_rcp;          // variables 0 .. k_rcp-1 have a reciprocal row (per pass)
    int k_un;           // variables 0 .. k_un-1 have their five unary rows staged in shared memory
    int slot_col0;      // first tensor-memory column of the slot blocks
    int tmem_slots;     // S_T: slots per warp held in tensor memory (the deeper ones are in local memory)
    int off_ys, off_meta, off_un, off_ring;   // shared-memory layout, byte offsets: y (and centred y), queue windows, unary rows, rings
    // a call with 513..1024 cases and the MSE fitness is SPLIT into one launch per pass of 512 cases: a launch then stages one
    // pass's variable rows, which leaves a slot row more per warp (half as many pushes go to local memory)
    int pass0, npass;   // first pass and number of passes this launch covers
    int un_w;           // cases per staged unary row: all padded cases, or 512 in a split call
    int ung_off;        // offset of this launch's rows in ung[]
    int pmode;          // 0: one launch does everything; 1 | 2: first | second launch of a split call (interp.cuh)
    float* partial;     // split call: the lanes' sums after pass 0, 32 floats per individual
};

// ---- PTX helpers: mbarrier, TMA bulk copy -----------------------------------------------------------
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

__host__ __device__ __forceinline__ int clamp_len(int l) { return (l >= 1 && l <= BEAGLE_MAX_LEN) ? l : 0; }
__device__ __host__ __forceinline__ int uop_stride(int len) { return (len + 3 + 1) & ~1; }   // records: n <= len micro-ops + 3; even

// The bodies of the three pre-pass kernels are prepass_body.inc; these are the device's meanings of its macros.
#define PB_SHARED(type, name, count) __shared__ type name[count];
#define PB_SHARED1(type, name) __shared__ type name;
#define PB_TID threadIdx.x
#define PB_BID blockIdx.x
#define PB_BDIM blockDim.x
#define PB_SYNC __syncthreads();
#define PB_SHFL_XOR(v, m) __shfl_xor_sync(0xffffffffu, v, m)
#define PB_SHFL_UP(v, s) __shfl_up_sync(0xffffffffu, v, s)
#define PB_ATOMIC_ADD(p, v) atomicAdd(p, v)
#define PB_ATOMIC_MAX(p, v) atomicMax(p, v)
#define PB_ATOMIC_OR(p, v) atomicOr(p, v)
#define PB_OP_SIN(v) op_sin(v)
#define PB_OP_COS(v) op_cos(v)
#define PB_OP_LOG(v) op_log(v)
#define PB_OP_SQRT(v) op_sqrt(v)
#define PB_OP_EXP(v) op_exp(v)
#define PB_U2F(u) __uint_as_float(u)
// ---- a2: block sums of the lengths + histogram of the lengths -----------------------------------------
__global__ void __launch_bounds__(kScanThreads) k_len_pass1(const int32_t* __restrict__ lengths, long long P,
                                                            long long* __restrict__ bsum, int* __restrict__ bins)
{
#define PB_SECTION 1
#include "prepass_body.inc"
#undef PB_SECTION
}

// one block: exclusive scan of the block sums in place; exclusive scan of the bins -> binstart[] (positions
// in perm[]) and binubase[] (micro-op entries); resets bins/cursors/header for the next use; and a4's
// transpose of the fitness cases into the variable-major, zero-padded block every interpreter CTA bulk-copies.
__global__ void __launch_bounds__(1024) k_len_pass2(long long* __restrict__ bsum, int nblocks, Header* __restrict__ hdr,
                                                    int* __restrict__ bins, int* __restrict__ cursor,
                                                    int* __restrict__ binstart, long long* __restrict__ binubase,
                                                    const float* __restrict__ X, const float* __restrict__ y,
                                                    int n, int d, int npad, float* __restrict__ xt, float* __restrict__ ung, int split)
{
#define PB_SECTION 2
#include "prepass_body.inc"
#undef PB_SECTION
}

// ---- a3: offsets and the counting sort by length ---------------------------------------------------------
__global__ void __launch_bounds__(kScanThreads) k_scatter(
    const int32_t* __restrict__ lengths, long long P, const long long* __restrict__ bsum,
    const int* __restrict__ binstart, int* __restrict__ cursor, long long* __restrict__ off,
    int* __restrict__ depth_out, float* __restrict__ fitness,
    float* __restrict__ outputs, int n_cases, const long long* __restrict__ binubase,
    int4* __restrict__ sched)
{
#define PB_SECTION 3
#include "prepass_body.inc"
#undef PB_SECTION
}

// debug only (beagle_debug_schedule): the sorted order as an index array; entries past the sorted ones are -1
__global__ void k_perm_from_sched(const int4* __restrict__ sched, const Header* __restrict__ hdr, long long P, int* __restrict__ perm)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P) perm[i] = i < hdr->n_sorted ? sched[i].x : -1;
}

// ---- a3/a5: the tree compiler ----------------------------------------------------------------------------
// in length-sorted order (k_scatter left each individual's start record: index, length, token offset, record base):
// well-formedness (D3), maximum stack depth, and the micro-ops of uop.cuh in the program's own evaluation
// order. acc always holds the topmost computed entry; the computed entry with c others below it that is not in acc
// sits in slot c (tensor memory while c < S_T, local memory beyond).
struct CompileParams {
    const uint32_t* genomes; const int4* sched;   // one start record per sorted position (k_scatter)
    const float* consts; long long n_consts; int d; int tmem_slots; int k_rcp; int k_un; int un_row_bytes;
    Header* hdr;
    uint2* uops; long long ucap; int4* meta; int* depth; int* slow_list; int* gen_list;
    float* fitness; float* outputs; int n_cases; int emit;
};

#include "compile_kernel.inc"

// ---- the interpreter kernel -----------------------------------------------------------------------------
#include "eval_kernel.inc"

// ---- prior art as a baseline, and the slow path: the paper's mapping ------------------------
// One block per individual, one thread per fitness case, a 32-entry per-thread stack in local
// memory, every thread decodes every token. The residuals go through shared memory so that warp 0
// can add them in the canonical order: results are bit-identical to the warp-per-individual kernels.
// With list != nullptr the blocks walk list[0..*count) (individuals whose micro-ops did not fit).
__global__ void __launch_bounds__(1024) k_eval_blockwise(
    const int32_t* __restrict__ genomes, const long long* __restrict__ off, const int32_t* __restrict__ lengths,
    const int* __restrict__ depth, const float* __restrict__ consts, const float* __restrict__ X,
    const float* __restrict__ y, int n, int d, float tax, float* __restrict__ fitness, float* __restrict__ outputs,
    const int* __restrict__ list, const int* __restrict__ count, long long P, int fit, float M, int power,
    const Header* __restrict__ hdr, int* __restrict__ h_f1)
{
    __shared__ float res[BEAGLE_MAX_N];
    // the last kernel of a call tells the host (pinned, mapped memory) how many programs used the f1 commands: the next
    // call picks its k_compile instantiation by it (no copy, no synchronisation)
    // (h_f1[0] programs with f1 commands, [1] programs k_compile_general had to take, [2] programs on the slow list: the
    // last two size the grids of those two kernels, which are launched whether their lists are empty or not)
    if (h_f1 && blockIdx.x == 0 && threadIdx.x == 0) { h_f1[0] = hdr->n_f1; h_f1[1] = hdr->n_general; h_f1[2] = hdr->n_slow; }
    bool y_finite = true;
    if (fit == BEAGLE_FIT_CORRELATION) y_finite = __syncthreads_and(threadIdx.x >= n || finite32(__ldg(y + threadIdx.x)));
    const long long total = list ? (long long)*count : P;
    for (long long idx = blockIdx.x; idx < total; idx += gridDim.x) {
        const long long p = list ? (long long)list[idx] : idx;
        if (depth[p] == 0) continue;               // malformed: NaN already written by the pre-pass
        const int len = lengths[p];
        const uint32_t* tok = reinterpret_cast<const uint32_t*>(genomes) + off[p];
        const int i = threadIdx.x;
        if (i < n) {
            float st[BEAGLE_MAX_STACK], var[BEAGLE_MAX_VARS];
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
                case OPC_SIGN: st[sp - 1] = op_sign(st[sp - 1]); break;
                case OPC_SQUARE: st[sp - 1] = op_square(st[sp - 1]); break;
                case OPC_CUBE: st[sp - 1] = op_cube(st[sp - 1]); break;
                case OPC_CBRT: st[sp - 1] = op_cbrt(st[sp - 1]); break;
                case OPC_TAN: st[sp - 1] = op_tan(st[sp - 1]); break;
                case OPC_ARCSIN: st[sp - 1] = op_arcsin(st[sp - 1]); break;
                case OPC_ARCCOS: st[sp - 1] = op_arccos(st[sp - 1]); break;
                case OPC_ARCTAN: st[sp - 1] = op_arctan(st[sp - 1]); break;
                case OPC_TANH: st[sp - 1] = op_tanh(st[sp - 1]); break;
                case OPC_POW: st[sp - 2] = op_pow(st[sp - 2], st[sp - 1]); --sp; break;
                case OPC_COPY: var[arg & 31u] = st[sp - 1]; break;
                case OPC_PASTE: st[sp++] = var[arg & 31u]; break;
                case OPC_DUP: st[sp] = st[sp - 1]; ++sp; break;
                case OPC_SWAP: { const float b = st[sp - 1]; st[sp - 1] = st[sp - 2]; st[sp - 2] = b; break; }
                case OPC_DEL: --sp; break;
                default: break;
                }
            }
            if (outputs) outputs[(size_t)p * n + i] = st[sp - 1];
            res[i] = fit == BEAGLE_FIT_CORRELATION ? st[sp - 1]
                   : fit == BEAGLE_FIT_STD ? std_reward(st[sp - 1], __ldg(y + i), M, __fdiv_rn(M, 11.f), power)
                   : (y ? __fsub_rn(st[sp - 1], __ldg(y + i)) : 0.f);
        }
        __syncthreads();
        if (threadIdx.x < 32 && fitness && fit == BEAGLE_FIT_CORRELATION) {       // f2: fit_corr.cuh, the layout of k_eval
            const int lane = threadIdx.x;
            CorrState cs = { 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0 };
            for (int c0 = 0; c0 < n; c0 += kCasesPerPass) {
                float fv[16], yv[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    const int ci = c0 + (k >> 2) * 128 + lane * 4 + (k & 3);
                    fv[k] = ci < n ? res[ci] : 0.f;
                    yv[k] = ci < n ? __ldg(y + ci) : 0.f;
                }
                corr_pass(fv, yv, c0, n, lane, y_finite, cs);
            }
            if (lane == 0) fitness[p] = corr_finish(cs, n, len, M, tax);
        } else if (threadIdx.x < 32 && fitness) {
            const int lane = threadIdx.x;
            float acc = 0.f;
            for (int m = 0; m * 128 < n; ++m)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int ci = m * 128 + lane * 4 + e;
                    if (ci < n) { const float r = res[ci]; acc = fit == BEAGLE_FIT_STD ? __fadd_rn(acc, r) : __fmaf_rn(r, r, acc); }
                }
#pragma unroll
            for (int m = 16; m >= 1; m >>= 1) acc = __fadd_rn(acc, __shfl_xor_sync(0xffffffffu, acc, m));
            if (lane == 0) fitness[p] = fit == BEAGLE_FIT_STD ? __fmaf_rn(-tax, (float)len, acc) : __fmaf_rn(tax, (float)len, __fdiv_rn(acc, (float)n));
        }
        __syncthreads();
    }
}

// ======================================================================================================
//                                        host side
// ======================================================================================================
struct Workspace {
    long long cap_P = 0, cap_U = 0;            // individuals / micro-op entries the workspace holds
    long long promised_P = 0, promised_T = 0;  // beagle_reserve: calls with P <= promised_P have T <= promised_T
    long long* off = nullptr; int* depth = nullptr; int4* meta = nullptr; int4* sched = nullptr;
    int* slow_list = nullptr; long long* bsum = nullptr; float* partial = nullptr;
    uint2* uops = nullptr;
    int* bins = nullptr; int* cursor = nullptr; int* binstart = nullptr; long long* binubase = nullptr;
    float* xt = nullptr; float* ung = nullptr; Header* hdr = nullptr; long long* h_T = nullptr; int* h_f1 = nullptr;
    unsigned long long* rank_hist = nullptr;   // beagle_rank's histogram when the caller wants none
    // chunked staging
    long long stage_bytes = 0; int stage_n = 0; unsigned char* stage[kStageBufsMax] = {};   // stage[0] owns the allocation
    float* stage_consts = nullptr; long long stage_consts_cap = 0;
    cudaStream_t copy_stream = nullptr; cudaEvent_t ev_copied[kStageBufsMax] = {}, ev_free[kStageBufsMax] = {};
    cudaEvent_t ev_k[2 * kProfMax] = {}; cudaEvent_t ev_p[kProfMax] = {}; int prof_n = 0; bool prof_this = false;
    int num_sms = 0; int smem_optin = 0; bool device_ok = false; bool inited = false; bool need_T_readback = false;
};
static Workspace g_ws;
static int32_t g_last_cuda = 0;
static int32_t g_launches = 0;
static int32_t g_profiling = 0;     // 0: off; n > 0: every n-th call is bracketed by events
static int32_t g_prof_calls = 0;
struct FitSel { int kind; float M; int power; };
static const FitSel kFitMse = { BEAGLE_FIT_MSE, 0.f, 1 };   // the fitness function is an argument all the way down, never state

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
    if (!w.device_ok) { w.inited = true; return BEAGLE_ERR_UNSUPPORTED; }
    CU(cudaFuncSetAttribute(k_eval<BEAGLE_FIT_MSE, true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval<BEAGLE_FIT_MSE, true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval<BEAGLE_FIT_MSE, true, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval<BEAGLE_FIT_MSE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval<BEAGLE_FIT_CORRELATION, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    CU(cudaFuncSetAttribute(k_eval<BEAGLE_FIT_STD, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, w.smem_optin));
    { uint32_t lut[kW2Size]; uint2 tt[kTok2Size]; make_walk2_tabs(lut, tt);
      CU(cudaMemcpyToSymbol(g_walk2_lut, lut, sizeof(lut))); CU(cudaMemcpyToSymbol(g_tok2, tt, sizeof(tt))); }
    CU(cudaMalloc(&w.bins, sizeof(int) * kNumBins));
    CU(cudaMalloc(&w.cursor, sizeof(int) * kNumBins));
    CU(cudaMemset(w.bins, 0, sizeof(int) * kNumBins));
    CU(cudaMemset(w.cursor, 0, sizeof(int) * kNumBins));
    CU(cudaMalloc(&w.binstart, sizeof(int) * kNumBins));
    CU(cudaMalloc(&w.binubase, sizeof(long long) * kNumBins));
    CU(cudaMalloc(&w.xt, sizeof(float) * (BEAGLE_MAX_D + 1) * BEAGLE_MAX_N));
    CU(cudaMalloc(&w.ung, sizeof(float) * 5 * BEAGLE_MAX_D * BEAGLE_MAX_N));
    CU(cudaMalloc(&w.hdr, sizeof(Header)));
    CU(cudaMemset(w.hdr, 0, sizeof(Header)));
    CU(cudaMallocHost(&w.h_T, sizeof(long long)));
    CU(cudaMallocHost(&w.h_f1, 4 * sizeof(int)));
    w.h_f1[0] = 0; w.h_f1[1] = 1; w.h_f1[2] = 1;   // the first call launches full grids
    w.inited = true;                               // only now: a failed allocation above is tried again by the next call
    return BEAGLE_OK;
}

static beagle_status reserve_P(long long P)
{
    Workspace& w = g_ws;
    if (P <= w.cap_P) return BEAGLE_OK;
    CU(cudaDeviceSynchronize());
    cudaFree(w.off); cudaFree(w.depth); cudaFree(w.meta); cudaFree(w.sched);
    cudaFree(w.slow_list); cudaFree(w.bsum); cudaFree(w.partial);
    w.off = nullptr; w.depth = nullptr; w.meta = nullptr; w.sched = nullptr;
    w.slow_list = nullptr; w.bsum = nullptr; w.partial = nullptr; w.cap_P = 0;
    (void)cudaGetLastError();                      // the frees are best effort: their status is not the call's
    const long long nb = (P + kScanBlock - 1) / kScanBlock;
    CU(cudaMalloc(&w.off, sizeof(long long) * (P + 1)));
    CU(cudaMalloc(&w.depth, sizeof(int) * P));
    CU(cudaMalloc(&w.sched, sizeof(int4) * P));
    CU(cudaMalloc(&w.meta, sizeof(int4) * P));
    CU(cudaMalloc(&w.slow_list, sizeof(int) * 2 * P));       // + the list of k_compile_general
    CU(cudaMalloc(&w.bsum, sizeof(long long) * (nb + 1)));
    CU(cudaMalloc(&w.partial, sizeof(float) * 32 * P));              // split calls (more than 512 cases): the lanes' sums after pass 0
    w.cap_P = P;
    return BEAGLE_OK;
}

static beagle_status reserve_U(long long U)
{
    Workspace& w = g_ws;
    if (U <= w.cap_U) return BEAGLE_OK;
    CU(cudaDeviceSynchronize());
    // meta[] and the TMA source address carry the record base in 16-byte units as 32 bits: 2^33 records (64 GiB)
    if (U > (1ll << 33)) return BEAGLE_ERR_UNSUPPORTED;
    cudaFree(w.uops); w.uops = nullptr; w.cap_U = 0;
    (void)cudaGetLastError();
    CU(cudaMalloc(&w.uops, sizeof(uint2) * U));
    w.cap_U = U;
    return BEAGLE_OK;
}

static long long uop_entries_bound(long long P, long long T) { return T + 4 * P + 2; }   // sum of uop_stride(len)

// a4's plan of the 512 tensor-memory columns (16 per row: a lane's 16 cases): the variable block (one row per
// variable and pass), the reciprocal rows of variables 0 .. k_rcp-1 (division by a variable becomes a
// multiplication, uop.cuh), then S_T slot rows for each warp of a lane quarter. The number of warps per
// quarter (8, 7 or 6: 1024, 896 or 768 threads) is chosen so that three slot rows per warp remain when
// possible. fast == false: the variable block alone does not fit (d > 32 at N <= 512, d > 16 beyond), and the
// call takes the blockwise kernel.
struct TmemPlan { bool split; bool fast; int threads; int rcp_col0; int k_rcp; int slot_col0; int tmem_slots; int k_un; int ring_bytes; size_t smem; int off_ys, off_meta, off_un, off_ring; };
static TmemPlan tmem_plan(int N, int d, int fit_kind, bool split)
{
    TmemPlan t = { split, false, kEvalThreads, 0, 0, 0, 0, 0, 0, 0 };
    const int passes = split ? 1 : (N + kCasesPerPass - 1) / kCasesPerPass;      // passes a launch stages
    const int rows = kTmemCols / kCasesPerLane;                  // 32
    const int xrows = passes * d;
    if (xrows > rows) return t;
    t.fast = true;
    const int wq_max = kEvalThreads / 128;
    // Slot rows come first (a slot beyond S_T costs local-memory traffic: config 4 runs 1.22x faster with two
    // slot rows per warp than with one plus reciprocal rows): S = the slot rows per warp that 6..8 warps per
    // quarter can have without reciprocal rows, at most 3. Among the plans that keep S, prefer 7 or 8 warps,
    // then the most reciprocal rows, then the most warps.
    const int free0 = rows - xrows;
    int S = 0;
    for (int c = 6; c <= wq_max; ++c) S = (free0 / c > S) ? free0 / c : S;
    S = S > 3 ? 3 : S;
    int wq = wq_max, k = 0, best = -1;
    for (int c = 6; c <= wq_max; ++c)
        for (int kk = 0; kk <= d; ++kk) {
            if (free0 - passes * kk < 0 || (free0 - passes * kk) / c < S) break;
            const int score = (c >= 7 ? 10000 : 0) + (c >= 8 ? BEAGLE_PLAN_W8 : 0) + kk * 10 + c;
            if (score > best) { best = score; wq = c; k = kk; }
        }
    const int free_rows = free0 - passes * k;
    int st = free_rows / wq;
    if (st > kMemSlots) st = kMemSlots;
    t.threads = wq * 128;
    t.rcp_col0 = xrows * kCasesPerLane; t.k_rcp = k;
    t.slot_col0 = (xrows + passes * k) * kCasesPerLane; t.tmem_slots = st;
    // shared memory: barriers, y, the warps' queue windows, then the staged rows f(X[j]) of the five unary commands
    // for variables 0 .. k_un-1 (a unary command on a variable is loop-invariant: uop.cuh H_LS), then the rings;
    // every warp keeps room for at least one stage of the longest program
    const int warps = t.threads / 32;
    const int npad = (N + kCasePad - 1) / kCasePad * kCasePad;
    const long long fixed = ((64 + warps * kStagesMax * 8 + 127) & ~127) + (long long)npad * 4 * (fit_kind == BEAGLE_FIT_CORRELATION ? 2 : 1)
                            + (long long)kEvalMetaBytes * warps;      // correlation: y and the centred y (eval_kernel.inc)
    const long long spare = (long long)g_ws.smem_optin - fixed - (long long)warps * ((kStageBytesMax + 127) & ~127);
    const int un_w = split ? kCasesPerPass : npad;
    long long ku = spare / (5ll * un_w * 4);
    t.k_un = (int)(ku < 0 ? 0 : (ku > d ? d : ku));
    const long long un_bytes = 5ll * t.k_un * un_w * 4;
    long long ring = ((g_ws.smem_optin - fixed - un_bytes) / warps) & ~127ll;
    if (ring > (long long)kStagesMax * kStageBytesMax) ring = (long long)kStagesMax * kStageBytesMax;
    t.ring_bytes = (int)ring;
    t.smem = (size_t)(fixed + un_bytes + ring * warps);
    t.off_ys = (64 + warps * kStagesMax * 8 + 127) & ~127;
    t.off_meta = (int)(fixed - (long long)kEvalMetaBytes * warps);
    t.off_un = (int)fixed; t.off_ring = (int)(fixed + un_bytes);
    return t;
}

// A call with 513..1024 cases that ends in the grouped MSE interpreter (no per-case outputs, no other fitness function) is
// split into one launch per pass (EvalParams::pmode); everything else stages all passes in one launch.
static TmemPlan plan_for(int N, int d, const FitSel& fit, bool mse_fitness_only)
{
    const TmemPlan whole = tmem_plan(N, d, fit.kind, false);
    if (!(N > kCasesPerPass && fit.kind == BEAGLE_FIT_MSE && mse_fitness_only)) return whole;
    // worth a second launch only where it buys slot rows (or makes the variable block fit at all): config 4's 9 variables
    // leave 2 slot rows per warp in one launch and 3 in two; config 2's 3 variables leave 3 either way
    const TmemPlan split = tmem_plan(N, d, fit.kind, true);
    return (!whole.fast || split.tmem_slots > whole.tmem_slots) ? split : whole;
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

// The only places where a call may block the host (include/beagle.h "Blocking"): the per-individual arrays grow when P
// exceeds what was ever reserved or used; the micro-op workspace grows when it is not known to hold the call. T_known < 0:
// the token count is not known on the host; the workspace is known to be enough when it holds the worst case, or when
// beagle_reserve promised a bound for colonies of this size; otherwise the token total is read back once, after the
// length scan of run_prepass (one cudaStreamSynchronize). Inside a stream capture nothing of this can be done: the call returns
// BEAGLE_ERR_NOT_RESERVED and enqueues nothing.
static bool is_capturing(cudaStream_t st)
{
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return cs != cudaStreamCaptureStatusNone;
}

static beagle_status ready_or_grow(long long P, long long T_known, bool emit, cudaStream_t st)
{
    Workspace& w = g_ws;
    const bool cap = is_capturing(st);
    if (P > w.cap_P) {
        if (cap) return BEAGLE_ERR_NOT_RESERVED;
        beagle_status s = reserve_P(P); if (s != BEAGLE_OK) return s;
    }
    if (!emit) return BEAGLE_OK;
    long long need = 0;
    if (T_known >= 0) need = uop_entries_bound(P, T_known);
    else if (w.cap_U >= (long long)uop_stride(BEAGLE_MAX_LEN) * P) need = 0;           // worst case fits
    else if (P <= w.promised_P && w.promised_T > 0) need = 0;                           // promised by beagle_reserve
    else need = -1;
    if (need == 0 || (need > 0 && need <= w.cap_U)) return BEAGLE_OK;
    if (cap) return BEAGLE_ERR_NOT_RESERVED;
    if (need < 0) { w.need_T_readback = true; return BEAGLE_OK; }                      // run_prepass reads it after its scan
    return reserve_U(need);
}

// a2 + a3 + the compile step of a5 (+ the transpose of a4). T_known < 0: the token count is not known
// on the host; unless beagle_reserve promised a bound, it is read back once (one stream synchronisation).
static beagle_status run_prepass(const int32_t* genomes, const int32_t* lengths, long long P, const float* consts,
                                 long long n_consts, const float* X, const float* y, int N, int d, float* fitness,
                                 float* outputs, long long T_known, bool emit, const FitSel& fit, cudaStream_t st)
{
    Workspace& w = g_ws;
    const int nb = (int)((P + kScanBlock - 1) / kScanBlock);
    const int npad = (N + kCasePad - 1) / kCasePad * kCasePad;
    // beagle_set_profiling: every n-th call is bracketed by events: pre-pass start, interpreter start, interpreter end
    w.prof_this = emit && g_profiling && w.prof_n < kProfMax && (g_prof_calls++ % g_profiling) == 0;
    if (w.prof_this) {
        if (!w.ev_p[w.prof_n]) CU(cudaEventCreate(&w.ev_p[w.prof_n]));
        CU(cudaEventRecord(w.ev_p[w.prof_n], st));
    }
    k_len_pass1<<<nb, kScanThreads, 0, st>>>(lengths, P, w.bsum, w.bins);
    k_len_pass2<<<1, 1024, 0, st>>>(w.bsum, nb, w.hdr, w.bins, w.cursor, w.binstart, w.binubase, X, y, N, d, npad, w.xt, w.ung, plan_for(N, d, fit, fitness && !outputs).split ? 1 : 0);
    g_launches += 2;
    if (emit && w.need_T_readback) {               // ready_or_grow: the one read-back of an un-reserved call
        w.need_T_readback = false;
        CU(cudaMemcpyAsync(w.h_T, &w.hdr->T, sizeof(long long), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        const long long need = uop_entries_bound(P, *w.h_T);
        if (need > w.cap_U) { beagle_status s = reserve_U(need); if (s != BEAGLE_OK) return s; }
    }
    k_scatter<<<nb, kScanThreads, 0, st>>>(lengths, P, w.bsum, w.binstart, w.cursor, w.off, w.depth,
                                           fitness, outputs, N, w.binubase, w.sched);
    ++g_launches;
    {
        CompileParams q;
        q.genomes = reinterpret_cast<const uint32_t*>(genomes); q.sched = w.sched;
        const TmemPlan tp = plan_for(N, d, fit, fitness && !outputs);
        q.consts = consts; q.n_consts = n_consts; q.d = d; q.tmem_slots = tp.tmem_slots; q.k_rcp = tp.k_rcp; q.k_un = tp.k_un; q.un_row_bytes = (tp.split ? kCasesPerPass : npad) * 4;
        q.hdr = w.hdr; q.uops = w.uops; q.ucap = w.cap_U; q.meta = w.meta; q.depth = w.depth;
        q.slow_list = w.slow_list; q.gen_list = w.slow_list + w.cap_P; q.fitness = fitness; q.outputs = outputs; q.n_cases = N; q.emit = emit ? 1 : 0;
        // the previous call's count of f1 programs, copied to pinned memory without a synchronisation: possibly stale, only a
        // guess at which instantiation is faster for this colony
        if (*w.h_f1 > 0) k_compile<true><<<(unsigned)((P + kCompileThreads - 1) / kCompileThreads), kCompileThreads, 0, st>>>(q);
        else k_compile<false><<<(unsigned)((P + kCompileThreads - 1) / kCompileThreads), kCompileThreads, 0, st>>>(q);
        long long gb = (P + kCompileThreads - 1) / kCompileThreads;
        // an empty list costs the launch of the blocks that would walk it (8 us at 16 per SM): a few blocks when the previous
        // call's list was empty (the grid strides over the list, so a wrong guess only moves time)
        const long long gcap = w.h_f1[1] > 0 ? (long long)w.num_sms * 8 : 8;
        k_compile_general<<<(unsigned)(gb > gcap ? gcap : gb), kCompileThreads, 0, st>>>(q);
        g_launches += 2;
    }
    CU(cudaGetLastError());
    return BEAGLE_OK;
}

static beagle_status run_eval(const int32_t* genomes, const int32_t* lengths, const float* consts, const float* X,
                              const float* y, long long P, int N, int d, float tax, float* fitness, float* outputs,
                              const FitSel& fit, cudaStream_t st)
{
    Workspace& w = g_ws;
    const int npad = (N + kCasePad - 1) / kCasePad * kCasePad;
    EvalParams prm;
    const TmemPlan tp = plan_for(N, d, fit, fitness && !outputs);
    if (!tp.fast) return BEAGLE_ERR_UNSUPPORTED;   // callers check first
    prm.rcp_col0 = tp.rcp_col0; prm.k_rcp = tp.k_rcp; prm.slot_col0 = tp.slot_col0; prm.tmem_slots = tp.tmem_slots;
    prm.meta = w.meta; prm.uops = w.uops; prm.hdr = w.hdr; prm.xt = w.xt; prm.ung = w.ung;
    prm.fitness = fitness; prm.outputs = outputs; prm.tax = tax; prm.M = fit.M; prm.power = fit.power; prm.n = N; prm.npad = npad; prm.d = d;
    const bool prof = w.prof_this;
    if (prof) {
        for (int i = 0; i < 2; ++i)
            if (!w.ev_k[2 * w.prof_n + i]) CU(cudaEventCreate(&w.ev_k[2 * w.prof_n + i]));
        CU(cudaEventRecord(w.ev_k[2 * w.prof_n], st));
    }
    const size_t smem = tp.smem;
    prm.ring_bytes = tp.ring_bytes; prm.k_un = tp.k_un;
    prm.off_ys = tp.off_ys; prm.off_meta = tp.off_meta; prm.off_un = tp.off_un; prm.off_ring = tp.off_ring;
    if (prm.ring_bytes < kStageBytesMax) return BEAGLE_ERR_UNSUPPORTED;
    prm.queue = &w.hdr->queue;
    const int passes_all = (N + kCasesPerPass - 1) / kCasesPerPass;
    prm.pass0 = 0; prm.npass = tp.split ? 1 : passes_all; prm.un_w = tp.split ? kCasesPerPass : npad; prm.ung_off = 0;
    prm.pmode = tp.split ? 1 : 0; prm.partial = w.partial;
    // programmatic dependent launch: k_eval's prologue (tensor-memory allocation, staging of X, y and the unary rows)
    // overlaps the tail of k_compile, which releases its dependents at its start; k_eval waits (griddepcontrol.wait)
    // before it touches the compiler's output
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(w.num_sms); cfg.blockDim = dim3(tp.threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (fit.kind == BEAGLE_FIT_CORRELATION) CU(cudaLaunchKernelEx(&cfg, k_eval<BEAGLE_FIT_CORRELATION, false>, prm));
    else if (fit.kind == BEAGLE_FIT_STD) CU(cudaLaunchKernelEx(&cfg, k_eval<BEAGLE_FIT_STD, false>, prm));
    else if (outputs || !fitness) CU(cudaLaunchKernelEx(&cfg, k_eval<BEAGLE_FIT_MSE, false>, prm));
    else if (tp.split) CU(cudaLaunchKernelEx(&cfg, k_eval<BEAGLE_FIT_MSE, true, 1>, prm));
    else CU(cudaLaunchKernelEx(&cfg, k_eval<BEAGLE_FIT_MSE, true, 0>, prm));
    ++g_launches;
    if (tp.split) {                                // the second pass: its own variable rows, the lanes' sums taken back
        prm.pass0 = 1; prm.pmode = 2; prm.ung_off = 5 * d * kCasesPerPass; prm.queue = &w.hdr->queue2;
        cfg.numAttrs = 0;
        CU(cudaLaunchKernelEx(&cfg, k_eval<BEAGLE_FIT_MSE, true, 2>, prm));
        ++g_launches;
    }
    if (prof) { CU(cudaEventRecord(w.ev_k[2 * w.prof_n + 1], st)); ++w.prof_n; }
    // slow path: individuals whose micro-ops did not fit the promised workspace (normally none)
    k_eval_blockwise<<<w.h_f1[2] > 0 ? w.num_sms * 2 : 4, (N + 31) / 32 * 32, 0, st>>>(genomes, w.off, lengths, w.depth, consts, X, y, N, d, tax,
                                                                   fitness, outputs, w.slow_list, &w.hdr->n_slow, P, fit.kind, fit.M, fit.power,
                                                                   w.hdr, w.h_f1);
    ++g_launches;
    CU(cudaGetLastError());
    return BEAGLE_OK;
}

// the whole path for one device-resident (chunk of a) colony: pre-pass + interpreter; when the variable
// block does not fit tensor memory, the pre-pass (as a well-formedness check) + the blockwise kernel,
// whose results are bit-identical (same per-command functions, same summation order).
static beagle_status run_colony(const int32_t* genomes, const int32_t* lengths, long long P, const float* consts,
                                long long n_consts, const float* X, const float* y, int N, int d, float tax,
                                float* fitness, float* outputs, long long T_known, const FitSel& fit, cudaStream_t st)
{
    Workspace& w = g_ws;
    const bool fast = plan_for(N, d, fit, fitness && !outputs).fast;
    beagle_status s = run_prepass(genomes, lengths, P, consts, n_consts, X, y, N, d, fitness, outputs, T_known, fast, fit, st);
    if (s != BEAGLE_OK) return s;
    if (fast) return run_eval(genomes, lengths, consts, X, y, P, N, d, tax, fitness, outputs, fit, st);
    k_eval_blockwise<<<(unsigned)P, (N + 31) / 32 * 32, 0, st>>>(genomes, w.off, lengths, w.depth, consts, X, y, N, d, tax,
                                                                fitness, outputs, nullptr, nullptr, P, fit.kind, fit.M, fit.power, nullptr, nullptr);
    ++g_launches;
    CU(cudaGetLastError());
    return BEAGLE_OK;
}

#include "simt_host.inc"

} // namespace beagle

using namespace beagle;

// BEAGLE_FIT_* of include/beagle.h -> kernel variant and power of the Std family
static bool decode_fit(int32_t fit, int* kind, int* power)
{
    *power = 1;
    switch (fit) {
    case BEAGLE_FIT_MSE: case BEAGLE_FIT_CORRELATION: *kind = fit; return true;
    case BEAGLE_FIT_STD: *kind = BEAGLE_FIT_STD; *power = 1; return true;
    case BEAGLE_FIT_STD_SQUARE: *kind = BEAGLE_FIT_STD; *power = 2; return true;
    case BEAGLE_FIT_STD_CUBE: *kind = BEAGLE_FIT_STD; *power = 3; return true;
    case BEAGLE_FIT_STD_HYPER: *kind = BEAGLE_FIT_STD; *power = 8; return true;
    default: return false;
    }
}

// ---- a8's host logic: how a budget is cut into staging buffers, and where a chunk ends (pure functions) -------------------
// The budget is cut into K staging buffers of about g_stage_target bytes (2 <= K <= 8), each a multiple of 256 bytes; false: a
// buffer could not hold one maximum-length individual.
static bool stage_layout(long long budget, long long* K_out, long long* bytes_out)
{
    long long K = budget / g_stage_target;
    K = K < 2 ? 2 : (K > kStageBufsMax ? kStageBufsMax : K);
    const long long half = (budget / K) & ~255ll;
    *K_out = K; *bytes_out = half;
    return half >= 4ll * (BEAGLE_MAX_LEN + 1);
}

// The chunk that starts at individual p0 ends before individual p1 (returned): as many whole individuals as fit cap_words
// words, one word per length plus one per token (a length outside 1..512 counts no tokens). *ntok: the chunk's tokens.
static long long chunk_end(const int32_t* h_lengths, long long P, long long p0, long long cap_words, long long* ntok_out)
{
    long long words = 0, p1 = p0, ntok = 0;
    // whole blocks of 4096 lengths first (a branch-free sum the host compiler vectorises: the scan of the first
    // chunk is on the critical path, nothing is in flight yet), then one by one up to the boundary
    while (p1 + 4096 <= P) {
        long long bt = 0;
        const int32_t* hl = h_lengths + p1;
        for (int k = 0; k < 4096; ++k) { const int32_t v = hl[k]; bt += (v >= 1 && v <= BEAGLE_MAX_LEN) ? v : 0; }
        if (words + bt + 4096 > cap_words) break;
        words += bt + 4096; ntok += bt; p1 += 4096;
    }
    while (p1 < P) {
        const int l = (h_lengths[p1] >= 1 && h_lengths[p1] <= BEAGLE_MAX_LEN) ? h_lengths[p1] : 0;
        if (words + l + 1 > cap_words) break;
        words += l + 1; ntok += l; ++p1;
    }
    *ntok_out = ntok;
    return p1;
}

static beagle_status eval_chunked_impl(const int32_t*, const int32_t*, int64_t, const float*, int64_t, const float*, const float*,
                                       int32_t, int32_t, float, float*, int64_t, const FitSel&, void*);

static beagle_status eval_impl(const int32_t* genomes, const int32_t* lengths, int64_t P,
                               const float* consts, int64_t n_consts, const float* X, const float* y,
                               int32_t N, int32_t d, float tax, float* fitness_out, const FitSel& fit, void* stream)
{
    beagle_status s = check_args(genomes, lengths, P, consts, n_consts, X, y, N, d, fitness_out);
    if (s != BEAGLE_OK) return s;
    g_launches = 0;
    if (P == 0) return BEAGLE_OK;
    if ((s = init_once()) != BEAGLE_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    if ((s = ready_or_grow(P, -1, plan_for(N, d, fit, true).fast, st)) != BEAGLE_OK) return s;
    return run_colony(genomes, lengths, P, consts, n_consts, X, y, N, d, tax, fitness_out, nullptr, -1, fit, st);
}

extern "C" {

beagle_status beagle_eval(const int32_t* genomes, const int32_t* lengths, int64_t P,
                          const float* consts, int64_t n_consts, const float* X, const float* y,
                          int32_t N, int32_t d, float tax, float* fitness_out, void* stream)
{
    return eval_impl(genomes, lengths, P, consts, n_consts, X, y, N, d, tax, fitness_out, kFitMse, stream);
}

beagle_status beagle_eval_fit(const int32_t* genomes, const int32_t* lengths, int64_t P,
                              const float* consts, int64_t n_consts, const float* X, const float* y,
                              int32_t N, int32_t d, int32_t fit, float M, float tax, float* fitness_out, void* stream)
{
    int kind, power;
    if (!decode_fit(fit, &kind, &power)) return BEAGLE_ERR_INVALID_ARG;
    const FitSel sel = { kind, M, power };
    return eval_impl(genomes, lengths, P, consts, n_consts, X, y, N, d, tax, fitness_out, sel, stream);
}

beagle_status beagle_rank(const float* fitness, int64_t P, const int64_t* sample_idx, int32_t n_sample,
                          int32_t maximise, uint8_t* decile_out, int64_t* hist_out, void* stream)
{
    if (P < 0 || n_sample < 1 || n_sample > kRankMaxSample) return BEAGLE_ERR_INVALID_ARG;
    if (P > 0 && (!fitness || !sample_idx || !decile_out)) return BEAGLE_ERR_INVALID_ARG;
    g_launches = 0;
    beagle_status s;
    if ((s = init_once()) != BEAGLE_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& w = g_ws;
    if (!w.rank_hist) CU(cudaMalloc(&w.rank_hist, 10 * sizeof(unsigned long long)));
    unsigned long long* hist = hist_out ? reinterpret_cast<unsigned long long*>(hist_out) : w.rank_hist;
    CU(cudaMemsetAsync(hist, 0, 10 * sizeof(unsigned long long), st));
    if (P == 0) return BEAGLE_OK;
    long long blocks = (P + kRankThreads * 8 - 1) / (kRankThreads * 8);
    const long long cap = (long long)w.num_sms * 8;
    blocks = blocks > cap ? cap : blocks;
    k_rank<<<(unsigned)blocks, kRankThreads, 0, st>>>(fitness, P, reinterpret_cast<const long long*>(sample_idx), n_sample,
                                                      maximise != 0, decile_out, hist);
    ++g_launches;
    CU(cudaGetLastError());
    return BEAGLE_OK;
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
    cudaStream_t st = (cudaStream_t)stream;
    if ((s = ready_or_grow(P, -1, plan_for(N, d, kFitMse, false).fast, st)) != BEAGLE_OK) return s;
    return run_colony(genomes, lengths, P, consts, n_consts, X, nullptr, N, d, 0.f, nullptr, out_PxN, -1, kFitMse, st);
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
    cudaStream_t st = (cudaStream_t)stream;
    if ((s = ready_or_grow(P, -1, false, st)) != BEAGLE_OK) return s;
    Workspace& w = g_ws;
    // k_compile runs as the well-formedness check only (depth[]); it emits no micro-ops
    if ((s = run_prepass(genomes, lengths, P, consts, n_consts, X, y, N, d, fitness_out, nullptr, -1, false, kFitMse, st)) != BEAGLE_OK) return s;
    const int threads = (N + 31) / 32 * 32;
    k_eval_blockwise<<<(unsigned)P, threads, 0, st>>>(genomes, w.off, lengths, w.depth, consts, X, y, N, d, tax,
                                                      fitness_out, nullptr, nullptr, nullptr, P, BEAGLE_FIT_MSE, 0.f, 1, nullptr, nullptr);
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
    if (perm && P > 0) {                           // the sorted order is the first word of the start records
        k_perm_from_sched<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(g_ws.sched, g_ws.hdr, P, perm);
        CU(cudaGetLastError());
    }
    return BEAGLE_OK;
}

beagle_status beagle_reserve_chunked(int64_t device_budget_bytes)
{
    Workspace& w = g_ws;
    beagle_status s = init_once();
    if (s != BEAGLE_OK) return s;
    // the budget is cut into K staging buffers of about 32 MiB (2 <= K <= 8): a chunk is copied while the ones before it
    // are evaluated, and the finer the chunks the less of the first copy and of the last evaluation is exposed
    long long K, half;
    if (!stage_layout(device_budget_bytes, &K, &half)) return BEAGLE_ERR_INVALID_ARG;
    if (!w.copy_stream) {
        CU(cudaStreamCreateWithFlags(&w.copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < kStageBufsMax; ++i) {
            CU(cudaEventCreateWithFlags(&w.ev_copied[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&w.ev_free[i], cudaEventDisableTiming));
        }
    }
    if (half != w.stage_bytes || (int)K != w.stage_n) {
        CU(cudaDeviceSynchronize());
        cudaFree(w.stage[0]); w.stage[0] = nullptr; w.stage_bytes = 0; w.stage_n = 0;
        CU(cudaMalloc(&w.stage[0], half * K));
        for (int i = 1; i < (int)K; ++i) w.stage[i] = w.stage[0] + (size_t)i * half;
        w.stage_bytes = half; w.stage_n = (int)K;
    }
    // workspace of one chunk: lengths + tokens fill at most cap_words words; an individual of L tokens takes at most
    // L + 4 records, and the most records per word come from one-token programs: 5 records for 2 words
    const long long cap_words = half / 4 - 3;
    if ((s = reserve_U(5 * cap_words / 2 + 4)) != BEAGLE_OK) return s;
    return BEAGLE_OK;
}

beagle_status beagle_eval_chunked_fit(const int32_t* h_genomes, const int32_t* h_lengths, int64_t P,
                                      const float* h_consts, int64_t n_consts, const float* X, const float* y,
                                      int32_t N, int32_t d, int32_t fit, float M, float tax, float* fitness_out,
                                      int64_t device_budget_bytes, void* stream)
{
    int kind, power;
    if (!decode_fit(fit, &kind, &power)) return BEAGLE_ERR_INVALID_ARG;
    const FitSel sel = { kind, M, power };
    return eval_chunked_impl(h_genomes, h_lengths, P, h_consts, n_consts, X, y, N, d, tax, fitness_out, device_budget_bytes, sel, stream);
}

beagle_status beagle_eval_chunked(const int32_t* h_genomes, const int32_t* h_lengths, int64_t P,
                                  const float* h_consts, int64_t n_consts, const float* X, const float* y,
                                  int32_t N, int32_t d, float tax, float* fitness_out,
                                  int64_t device_budget_bytes, void* stream)
{
    return eval_chunked_impl(h_genomes, h_lengths, P, h_consts, n_consts, X, y, N, d, tax, fitness_out, device_budget_bytes, kFitMse, stream);
}

} // extern "C"

static beagle_status eval_chunked_impl(const int32_t* h_genomes, const int32_t* h_lengths, int64_t P,
                                       const float* h_consts, int64_t n_consts, const float* X, const float* y,
                                       int32_t N, int32_t d, float tax, float* fitness_out,
                                       int64_t device_budget_bytes, const FitSel& fit, void* stream)
{
    beagle_status s = check_args(h_genomes, h_lengths, P, h_consts, n_consts, X, y, N, d, fitness_out);
    if (s != BEAGLE_OK) return s;
    if (device_budget_bytes < 2ll * 4 * (BEAGLE_MAX_LEN + 64)) return BEAGLE_ERR_INVALID_ARG;   // 4608: include/beagle.h
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
    for (int i = 1; i < w.stage_n; ++i) CU(cudaEventRecord(w.ev_free[i], st));
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
        long long ntok = 0;
        const long long p1 = chunk_end(h_lengths, P, p0, cap_words, &ntok);
        const long long np = p1 - p0;
        const int b = c % w.stage_n;
        int32_t* d_len = reinterpret_cast<int32_t*>(w.stage[b]);
        int32_t* d_tok = d_len + ((np + 3) & ~3ll);
        CU(cudaStreamWaitEvent(w.copy_stream, w.ev_free[b], 0));      // buffer b is free again
        CU(cudaMemcpyAsync(d_len, h_lengths + p0, sizeof(int32_t) * np, cudaMemcpyHostToDevice, w.copy_stream));
        if (ntok > 0)
            CU(cudaMemcpyAsync(d_tok, h_genomes + tok0, sizeof(int32_t) * ntok, cudaMemcpyHostToDevice, w.copy_stream));
        CU(cudaEventRecord(w.ev_copied[b], w.copy_stream));
        CU(cudaStreamWaitEvent(st, w.ev_copied[b], 0));
        if ((s = ready_or_grow(np, ntok, plan_for(N, d, fit, true).fast, st)) != BEAGLE_OK) return s;     // (reserved: a no-op)
        if ((s = run_colony(d_tok, d_len, np, w.stage_consts, n_consts, X, y, N, d, tax, fitness_out + p0, nullptr, ntok, fit, st)) != BEAGLE_OK) return s;
        CU(cudaEventRecord(w.ev_free[b], st));
        total_launches += g_launches; g_launches = 0;
        p0 = p1; tok0 += ntok;
    }
    g_launches = total_launches;
    return BEAGLE_OK;
}

extern "C" {

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
    case BEAGLE_ERR_NOT_RESERVED: return "the workspace would have to grow inside a stream capture: call beagle_reserve first";
    default: return "unknown status";
    }
}

int32_t beagle_last_cuda_error(void) { return g_last_cuda; }

beagle_status beagle_reserve(int64_t P_max, int64_t T_max)
{
    if (P_max < 0 || P_max > 0x7FFFFFFFll || T_max < 0) return BEAGLE_ERR_INVALID_ARG;
    beagle_status s = init_once();
    if (s != BEAGLE_OK) return s;
    if ((s = reserve_P(P_max)) != BEAGLE_OK) return s;
    if (T_max > 0) {
        if ((s = reserve_U(uop_entries_bound(P_max, T_max))) != BEAGLE_OK) return s;
        g_ws.promised_P = P_max; g_ws.promised_T = T_max;
    }
    return BEAGLE_OK;
}

void beagle_release(void)
{
    Workspace& w = g_ws;
    cudaDeviceSynchronize();
    cudaFree(w.off); cudaFree(w.depth); cudaFree(w.meta); cudaFree(w.sched);
    cudaFree(w.slow_list); cudaFree(w.bsum); cudaFree(w.uops); cudaFree(w.partial); w.partial = nullptr;
    cudaFree(w.stage[0]); cudaFree(w.stage_consts); cudaFree(w.rank_hist); w.rank_hist = nullptr;
    (void)cudaGetLastError();
    w.off = nullptr; w.depth = nullptr; w.meta = nullptr; w.sched = nullptr;
    w.slow_list = nullptr; w.bsum = nullptr; w.uops = nullptr; w.cap_P = 0; w.cap_U = 0;
    w.promised_P = 0; w.promised_T = 0;
    w.stage[0] = nullptr; w.stage_bytes = 0; w.stage_n = 0; w.stage_consts = nullptr; w.stage_consts_cap = 0;
}

int32_t beagle_last_launch_count(void) { return g_launches; }

// host only, no device needed: the plan of the 32 tensor-memory rows and of shared memory a call with these arguments would
// get on a device with smem_optin bytes of opt-in shared memory per block
beagle_status beagle_debug_plan(int32_t N, int32_t d, int32_t fit, int32_t fitness_only, int32_t smem_optin, int32_t* out12)
{
    int kind, power;
    if (!out12 || !decode_fit(fit, &kind, &power) || N < 1 || N > BEAGLE_MAX_N || d < 1 || d > BEAGLE_MAX_D || smem_optin < 0)
        return BEAGLE_ERR_INVALID_ARG;
    const FitSel sel = { kind, 0.f, power };
    const int saved = g_ws.smem_optin;
    g_ws.smem_optin = smem_optin;
    const TmemPlan tp = plan_for(N, d, sel, fitness_only != 0);
    g_ws.smem_optin = saved;
    const int passes = tp.split ? 1 : (N + kCasesPerPass - 1) / kCasesPerPass;
    const int v[12] = { tp.fast ? 1 : 0, tp.split ? 1 : 0, tp.threads, passes * d, passes * tp.k_rcp, tp.tmem_slots, tp.k_un, tp.ring_bytes,
                        (int)tp.smem, tp.off_ys, tp.off_un, tp.off_ring };
    for (int i = 0; i < 12; ++i) out12[i] = v[i];
    return BEAGLE_OK;
}

// host only: the chunks beagle_eval_chunked would cut this colony into under this budget (the same two functions)
beagle_status beagle_debug_chunk_plan(const int32_t* h_lengths, int64_t P, int64_t device_budget_bytes, int64_t* ends, int64_t max_ends,
                                      int64_t* n_chunks, int32_t* n_buffers, int64_t* buffer_bytes)
{
    if (P < 0 || (P > 0 && !h_lengths) || device_budget_bytes < 2ll * 4 * (BEAGLE_MAX_LEN + 64)) return BEAGLE_ERR_INVALID_ARG;
    long long K, half;
    if (!stage_layout(device_budget_bytes, &K, &half)) return BEAGLE_ERR_INVALID_ARG;
    if (n_buffers) *n_buffers = (int32_t)K;
    if (buffer_bytes) *buffer_bytes = half;
    const long long cap_words = half / 4 - 3;
    long long n = 0;
    for (long long p0 = 0; p0 < P; ++n) {
        long long ntok = 0;
        const long long p1 = chunk_end(h_lengths, P, p0, cap_words, &ntok);
        if (p1 == p0) return BEAGLE_ERR_INVALID_ARG;      // (cannot happen: a buffer holds a maximum-length individual)
        if (ends && n < max_ends) ends[n] = p1;
        p0 = p1;
    }
    if (n_chunks) *n_chunks = n;
    return BEAGLE_OK;
}

// host only: the two tables of the tree compiler's walk as the device gets them (compile_kernel.inc: make_walk2_tabs)
void beagle_debug_walk_tables(uint32_t* lut160, uint32_t* tok130)
{
    uint32_t lut[kW2Size]; uint2 tt[kTok2Size];
    make_walk2_tabs(lut, tt);
    if (lut160) for (int i = 0; i < kW2Size; ++i) lut160[i] = lut[i];
    if (tok130) for (int i = 0; i < kTok2Size; ++i) { tok130[2 * i] = tt[i].x; tok130[2 * i + 1] = tt[i].y; }
}

// host only: std_reward (fit_std.cuh), the reward of one (output, target) pair of the Std family, compiled for the host
beagle_status beagle_debug_std_reward(const float* f, const float* y, int64_t n, int32_t fit, float M, float* out)
{
    int kind, power;
    if (n < 0 || (n > 0 && (!f || !y || !out)) || !decode_fit(fit, &kind, &power) || kind != BEAGLE_FIT_STD) return BEAGLE_ERR_INVALID_ARG;
    const float pen = M / 11.f;                   // the kernels' __fdiv_rn(M, 11.f)
    for (int64_t i = 0; i < n; ++i) out[i] = std_reward(f[i], y[i], M, pen, power);
    return BEAGLE_OK;
}

// host only: the correlation fitness of ONE individual from its per-case outputs, by the functions of fit_corr.cuh on an emulated warp
beagle_status beagle_debug_corr(const float* f, const float* y, int32_t N, int32_t len, float M, float tax, int32_t pre, float* fitness_out)
{
    if (!f || !y || !fitness_out || N < 1 || N > BEAGLE_MAX_N || len < 1 || len > BEAGLE_MAX_LEN) return BEAGLE_ERR_INVALID_ARG;
    alignas(16) float dys[BEAGLE_MAX_N] = {};
    CorrYPass ypre[2] = {};
    float out = 0.f;
    try {
        if (!simt::run_block(32, 0, [&](simt::Block& blk, int tid) { h_corr_lane(blk, tid, f, y, N, len, M, tax, pre, dys, ypre, &out); }))
            return BEAGLE_ERR_UNSUPPORTED;
    } catch (...) { return BEAGLE_ERR_NOMEM; }
    *fitness_out = out;
    return BEAGLE_OK;
}

// host only: k_rank (rank_body.inc) run by the SIMT emulator, `grid` blocks one after the other
beagle_status beagle_debug_rank(const float* fitness, int64_t P, const int64_t* sample_idx, int32_t n_sample, int32_t maximise,
                                int32_t grid, uint8_t* decile_out, int64_t* hist_out)
{
    if (P < 1 || P > (1 << 22) || n_sample < 1 || n_sample > kRankMaxSample || grid < 1 || grid > 4096 || !fitness || !sample_idx
        || !decile_out || !hist_out)
        return BEAGLE_ERR_INVALID_ARG;
    for (int i = 0; i < n_sample; ++i) if (sample_idx[i] < 0 || sample_idx[i] >= P) return BEAGLE_ERR_INVALID_ARG;
    unsigned long long hist[10] = {};              // (beagle_rank zeroes the histogram before the launch)
    try {
    for (int b = 0; b < grid; ++b)
        if (!simt::run_block(kRankThreads, b, [&](simt::Block& blk, int tid) {
                h_rank(blk, tid, grid, fitness, P, reinterpret_cast<const long long*>(sample_idx), n_sample, maximise != 0, decile_out, hist); }))
            return BEAGLE_ERR_UNSUPPORTED;
    } catch (...) { return BEAGLE_ERR_NOMEM; }
    for (int i = 0; i < 10; ++i) hist_out[i] = (int64_t)hist[i];
    return BEAGLE_OK;
}

// host only: the pre-pass kernels k_len_pass1, k_len_pass2, k_scatter (prepass_body.inc) run by the SIMT emulator of simt_host.inc
beagle_status beagle_debug_prepass(const int32_t* lengths, int64_t P, const float* X, const float* y, int32_t N, int32_t d, int32_t split,
                                   int64_t* off, int32_t* sched4, float* fitness, int32_t* depth, float* xt, int64_t* hdr6,
                                   int32_t* binstart, int64_t* binubase)
{
    if (P < 1 || P > (1 << 24) || !lengths || !X || !y || N < 1 || N > BEAGLE_MAX_N || d < 1 || d > BEAGLE_MAX_D
        || !off || !sched4 || !fitness || !depth || !xt || !hdr6 || !binstart || !binubase)
        return BEAGLE_ERR_INVALID_ARG;
    try {                                          // (host containers inside: no exception may cross the C boundary)
    const int npad = (N + kCasePad - 1) / kCasePad * kCasePad;
    std::vector<float> ung((size_t)5 * d * npad, 0.f);
    Header hdr = {};
    static_assert(sizeof(long long) == sizeof(int64_t), "off and binubase are passed through as they are");
    if (!prepass_host(lengths, P, X, y, N, d, split ? 1 : 0, reinterpret_cast<long long*>(off), reinterpret_cast<int4*>(sched4), fitness, depth, xt,
                      ung.data(), &hdr, binstart, reinterpret_cast<long long*>(binubase)))
        return BEAGLE_ERR_UNSUPPORTED;             // the host gave the emulator no 1024 threads
    hdr6[0] = hdr.T; hdr6[1] = hdr.uop_entries; hdr6[2] = hdr.n_sorted; hdr6[3] = hdr.max_len; hdr6[4] = hdr.rcp_unsafe;
    hdr6[5] = hdr.n_malformed;                     // 0, or -1 if the length histogram was not left zeroed for the next call
    return BEAGLE_OK;
    } catch (...) { return BEAGLE_ERR_NOMEM; }
}

// host only: one warp of k_eval's scheduling loop (queue_body.inc) over a given list of queue entries, as a list of events
beagle_status beagle_debug_queue(const int32_t* meta4, int32_t total, int32_t max_len, int32_t ring_bytes, int32_t grid, int32_t threads,
                                 int32_t grouped, uint32_t skip_seed, uint32_t queue_start, int32_t* events, int32_t cap,
                                 int32_t* n_events, int32_t* sizing3)
{
    if (total < 0 || (total > 0 && !meta4) || max_len < 1 || max_len > BEAGLE_MAX_LEN || ring_bytes < kStageBytesMax || grid < 1
        || threads < 32 || threads > 1024 || (threads & 31) || cap < 0 || (cap > 0 && !events) || !n_events || !sizing3)
        return BEAGLE_ERR_INVALID_ARG;
    QueueLog L = { events, cap, 0 };
    unsigned int queue = queue_start;
    if (total > 0) {                               // (k_eval returns at once when nothing is sorted)
        if (grouped) queue_host<true>(reinterpret_cast<const int4*>(meta4), total, max_len, ring_bytes, grid, threads, &queue, skip_seed, L, sizing3);
        else queue_host<false>(reinterpret_cast<const int4*>(meta4), total, max_len, ring_bytes, grid, threads, &queue, skip_seed, L, sizing3);
    } else { sizing3[0] = sizing3[1] = sizing3[2] = 0; }
    *n_events = L.n;
    return BEAGLE_OK;
}

// host only: the body of k_compile's walk (walk_body.inc) on one program
beagle_status beagle_debug_walk(const int32_t* tokens, int32_t len, const float* consts, int64_t n_consts, int32_t d,
                                int32_t tmem_slots, int32_t k_rcp, int32_t k_un, int32_t un_row_bytes, uint32_t rcp_unsafe, int32_t f1,
                                uint32_t* records, int32_t* n_records, int32_t* depth, int32_t* taken, int32_t* used_f1)
{
    if (!tokens || len < 1 || len > BEAGLE_MAX_LEN || d < 1 || d > BEAGLE_MAX_D || n_consts < 0 || n_consts > BEAGLE_MAX_CONSTS
        || (n_consts > 0 && !consts) || tmem_slots < 0 || tmem_slots > kMemSlots || k_rcp < 0 || k_rcp > d || k_un < 0 || k_un > d
        || un_row_bytes < 0 || !records || !n_records || !depth || !taken || !used_f1)
        return BEAGLE_ERR_INVALID_ARG;
    Header hdr = {}; hdr.rcp_unsafe = rcp_unsafe;
    uint2 uops[BEAGLE_MAX_LEN + 8] = {};
    int4 meta[1] = {}; int dep[1] = { 0 }; int gen_list[1] = { -1 }, slow_list[1] = { -1 };
    CompileParams q = {};
    q.genomes = reinterpret_cast<const uint32_t*>(tokens);
    q.consts = consts; q.n_consts = n_consts; q.d = d; q.tmem_slots = tmem_slots; q.k_rcp = k_rcp; q.k_un = k_un; q.un_row_bytes = un_row_bytes;
    q.hdr = &hdr; q.uops = uops; q.ucap = BEAGLE_MAX_LEN + 8; q.meta = meta; q.depth = dep; q.slow_list = slow_list; q.gen_list = gen_list;
    q.emit = 1;
    const int mode = f1 & 0xff, longer = (f1 >> 8) & 0x3ff;      // f1 bits 17:8: a neighbouring lane's program is that much longer
    if (mode) walk_host<true>(q, len, mode == 2, longer); else walk_host<false>(q, len, false, longer);
    *taken = hdr.n_general == 0 ? 1 : 0;
    *depth = *taken ? dep[0] : 0;
    *used_f1 = hdr.n_f1;
    int n = 0;
    if (*taken) { while (n < BEAGLE_MAX_LEN + 4 && (uops[n].x & 255u) != H_END) ++n; }
    *n_records = n;
    for (int k = 0; k < n; ++k) { records[2 * k] = uops[k].x; records[2 * k + 1] = uops[k].y; }
    return BEAGLE_OK;
}

// host only: compile_general (compile_kernel.inc), the compiler of the whole language that k_compile_general runs one lane per
// program, compiled for the host and run on one program
beagle_status beagle_debug_compile(const int32_t* tokens, int32_t len, const float* consts, int64_t n_consts, int32_t d,
                                   int32_t tmem_slots, int32_t k_rcp, int32_t k_un, int32_t un_row_bytes, uint32_t rcp_unsafe,
                                   uint32_t* records, int32_t* n_records, int32_t* depth, int32_t* slow)
{
    if (!tokens || len < 1 || len > BEAGLE_MAX_LEN || d < 1 || d > BEAGLE_MAX_D || n_consts < 0 || n_consts > BEAGLE_MAX_CONSTS
        || (n_consts > 0 && !consts) || tmem_slots < 0 || tmem_slots > kMemSlots || k_rcp < 0 || k_rcp > d || k_un < 0 || k_un > d
        || un_row_bytes < 0 || !records || !n_records || !depth || !slow)
        return BEAGLE_ERR_INVALID_ARG;
    CompileParams q = {};
    q.consts = consts; q.n_consts = n_consts; q.d = d; q.tmem_slots = tmem_slots; q.k_rcp = k_rcp; q.k_un = k_un; q.un_row_bytes = un_row_bytes;
    const uint32_t rcp_ok = ~rcp_unsafe & ((k_rcp >= 32) ? 0xFFFFFFFFu : ((1u << k_rcp) - 1u));       // as the kernels form it
    uint2 out[BEAGLE_MAX_LEN + 4];
    int n = 0; bool sl = false;
    const int mx = compile_general(q, reinterpret_cast<const uint32_t*>(tokens), len, out, true, rcp_ok, &n, &sl);
    *depth = mx; *slow = (mx > 0 && sl) ? 1 : 0; *n_records = (mx > 0 && !sl) ? n : 0;
    if (mx > 0 && !sl) for (int i = 0; i < n; ++i) { records[2 * i] = out[i].x; records[2 * i + 1] = out[i].y; }
    return BEAGLE_OK;
}

beagle_status beagle_debug_counts(int32_t* n_sorted, int32_t* n_general, int32_t* n_slow, int32_t* n_malformed, void* stream)
{
    Header h;
    if (!g_ws.hdr) return BEAGLE_ERR_INVALID_ARG;
    CU(cudaMemcpyAsync(&h, g_ws.hdr, sizeof(Header), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    if (n_sorted) *n_sorted = h.n_sorted;
    if (n_general) *n_general = h.n_general;
    if (n_slow) *n_slow = h.n_slow;
    if (n_malformed) *n_malformed = h.n_malformed;
    return BEAGLE_OK;
}

void beagle_set_chunk_target(int64_t bytes) { g_stage_target = bytes > 0 ? bytes : kStageTarget; }

int32_t beagle_chunk_buffers(void) { return g_ws.stage_n; }

void beagle_set_profiling(int32_t on) { g_profiling = on < 0 ? 0 : on; g_prof_calls = 0; if (on) g_ws.prof_n = 0; }

float beagle_profiled_prepass_ms(int32_t* n_calls)
{
    Workspace& w = g_ws;
    if (n_calls) *n_calls = 0;
    if (w.prof_n <= 0) return -1.f;
    double sum = 0.0;
    for (int i = 0; i < w.prof_n; ++i) {
        float ms = 0.f;
        if (cudaEventSynchronize(w.ev_k[2 * i]) != cudaSuccess) return -1.f;
        if (cudaEventElapsedTime(&ms, w.ev_p[i], w.ev_k[2 * i]) != cudaSuccess) return -1.f;
        sum += ms;
    }
    if (n_calls) *n_calls = w.prof_n;
    return (float)(sum / w.prof_n);
}

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
