// probe_tmem_operand.cu — standalone measurement behind DESIGN.md §7 "tensor memory as the operand store"
// (not part of libbeagle_b200.so). A lane's 16 fitness cases of one variable fetched (a) by one
// tcgen05.ld.32x32b.x16 from tensor memory, (b) by 4 x LDS.128 from shared memory, each followed by 16 FADDs,
// for 1..32 warps per SM on all 148 SMs. Results: profiles/r1_probe_tmem_operand.md.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o probe_tmem_operand probe_tmem_operand.cu && ./probe_tmem_operand
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#define LD16(R, addr) asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];" \
    : "=f"(R[0]),"=f"(R[1]),"=f"(R[2]),"=f"(R[3]),"=f"(R[4]),"=f"(R[5]),"=f"(R[6]),"=f"(R[7]),"=f"(R[8]),"=f"(R[9]),"=f"(R[10]),"=f"(R[11]),"=f"(R[12]),"=f"(R[13]),"=f"(R[14]),"=f"(R[15]) : "r"(addr))
#define ST16(R, addr) asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%16], {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15};" \
    :: "f"(R[0]),"f"(R[1]),"f"(R[2]),"f"(R[3]),"f"(R[4]),"f"(R[5]),"f"(R[6]),"f"(R[7]),"f"(R[8]),"f"(R[9]),"f"(R[10]),"f"(R[11]),"f"(R[12]),"f"(R[13]),"f"(R[14]),"f"(R[15]), "r"(addr))

// mode 0: TMEM x16 + wait + 16 FADD ; mode 1: 4x LDS.128 + 16 FADD ; mode 2: TMEM, 2 loads in flight; mode 3: half TMEM half LDS alternate
__global__ void __launch_bounds__(1024, 1) k(int mode, int iters, float* out, long long* cyc, int check)
{
    __shared__ uint32_t tbase;
    extern __shared__ __align__(16) float xs[];      // 32 rows x 512 cases (row-major, lane*4.. layout like the interpreter)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 32 * 512; i += blockDim.x) xs[i] = (float)(i % 977) * 0.001f;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" :: "r"((uint32_t)__cvta_generic_to_shared(&tbase)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tb = tbase + ((uint32_t)(32 * (warp & 3)) << 16);
    if (warp < 4) {   // fill: row r -> columns [16r, 16r+16): value = xs[r*512 + g*128 + lane*4 + e], k = 4g+e
        for (int r = 0; r < 32; ++r) {
            float v[16];
            for (int kq = 0; kq < 16; ++kq) v[kq] = xs[r * 512 + (kq >> 2) * 128 + lane * 4 + (kq & 3)];
            ST16(v, tb + 16 * r);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    float acc[16];
    for (int kq = 0; kq < 16; ++kq) acc[kq] = 0.f;
    unsigned row = warp * 7u + 3u;
    long long t0 = clock64();
    if (mode == 0) {
        for (int it = 0; it < iters; ++it) {
            float x[16];
            row = (row * 5u + 1u) & 31u;
            LD16(x, tb + 16 * row);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int kq = 0; kq < 16; ++kq) acc[kq] += x[kq];
        }
    } else if (mode == 1) {
        for (int it = 0; it < iters; ++it) {
            row = (row * 5u + 1u) & 31u;
            const float4* p = reinterpret_cast<const float4*>(xs + row * 512 + lane * 4);
#pragma unroll
            for (int g = 0; g < 4; ++g) { float4 v = p[g * 32]; acc[4*g] += v.x; acc[4*g+1] += v.y; acc[4*g+2] += v.z; acc[4*g+3] += v.w; }
        }
    } else if (mode == 2) {
        float x[16], z[16];
        row = (row * 5u + 1u) & 31u;
        LD16(x, tb + 16 * row);
        for (int it = 0; it < iters; it += 2) {
            row = (row * 5u + 1u) & 31u;
            LD16(z, tb + 16 * row);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int kq = 0; kq < 16; ++kq) acc[kq] += x[kq];
            row = (row * 5u + 1u) & 31u;
            LD16(x, tb + 16 * row);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int kq = 0; kq < 16; ++kq) acc[kq] += z[kq];
        }
    } else if (mode == 3) {
        for (int it = 0; it < iters; it += 2) {
            float x[16];
            row = (row * 5u + 1u) & 31u;
            LD16(x, tb + 16 * row);
            row = (row * 5u + 1u) & 31u;
            const float4* p = reinterpret_cast<const float4*>(xs + row * 512 + lane * 4);
#pragma unroll
            for (int g = 0; g < 4; ++g) { float4 v = p[g * 32]; acc[4*g] += v.x; acc[4*g+1] += v.y; acc[4*g+2] += v.z; acc[4*g+3] += v.w; }
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int kq = 0; kq < 16; ++kq) acc[kq] += x[kq];
        }
    }
    long long t1 = clock64();
    float s = 0; for (int kq = 0; kq < 16; ++kq) s += acc[kq] * (kq + 1);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (lane == 0) cyc[blockIdx.x * (blockDim.x / 32) + warp] = t1 - t0;
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tbase));
}
int main()
{
    float* out; long long* cyc; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 148 * 32 * 8);
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 32 * 512 * 4);
    const char* names[] = {"TMEM x16 +wait +16 FADD", "4x LDS.128 +16 FADD", "TMEM x16 prefetch 1 ahead", "alternate TMEM / LDS"};
    float ref[4][2];
    for (int mode = 0; mode < 4; ++mode) for (int warps = 1; warps <= 32; warps *= 2) {
        if (warps == 2 || warps == 8) continue;
        const int iters = 4096;
        k<<<148, warps * 32, 32 * 512 * 4>>>(mode, iters, out, cyc, 0);
        cudaError_t e = cudaDeviceSynchronize();
        long long hc[148 * 32]; cudaMemcpy(hc, cyc, 148 * warps * 8, cudaMemcpyDeviceToHost);
        float ho[64]; cudaMemcpy(ho, out, 64 * 4, cudaMemcpyDeviceToHost);
        double avg = 0; long long mx = 0; for (int i = 0; i < 148 * warps; ++i) { avg += hc[i]; if (hc[i] > mx) mx = hc[i]; } avg /= 148 * warps;
        printf("%-28s warps=%2d cycles/iter per warp %.1f | loads/clk/SM %.4f  B/clk/SM %.0f  out[5]=%g out[37]=%g (%s)\n", names[mode], warps, avg / iters,
               warps * (double)iters / mx, warps * (double)iters / mx * 2048, ho[5], ho[37], cudaGetErrorString(e));
    }
    return 0;
}
