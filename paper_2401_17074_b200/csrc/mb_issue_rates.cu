// mb_issue_rates.cu -- stand-alone micro-benchmark behind the issue-rate figures quoted in DESIGN.md "Kernels" and
// profiles/README.md (not part of libtslb.so): how many cycles does a sub-partition of a B200 SM need per packed FFMA2,
// per scalar FFMA, and per FFMA2 paired with one instruction of another pipe (ALU, shuffle, shared load / store)?
// 148 CTAs x 16 warps (4 per sub-partition), 8 independent chains per thread, clock64 around 2000 x 32 slots.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o mb_issue_rates paper_2401_17074_b200/csrc/mb_issue_rates.cu && ./mb_issue_rates
#include <cstdio>
#include <cuda_runtime.h>
template <int MODE>
__global__ void __launch_bounds__(512, 1) k(float *out, int iters, long long *cyc)
{
    float2 a[8]; unsigned u[8]; float f[8];
    __shared__ float sm[2048];
    sm[threadIdx.x] = threadIdx.x; sm[threadIdx.x + 512] = 1.f; sm[threadIdx.x + 1024] = 1.f; sm[threadIdx.x + 1536] = 1.f;
    __syncthreads();
    unsigned sbase = (unsigned)__cvta_generic_to_shared(sm) + (threadIdx.x & 31) * 4;
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = make_float2(threadIdx.x * 0.001f + i, i * 0.5f); u[i] = threadIdx.x * 7 + i; f[i] = i + threadIdx.x; }
    const float2 m = make_float2(1.0001f, 0.9999f), c = make_float2(0.001f, -0.001f);
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE != 1 && MODE != 8 && MODE != 9) a[i] = __ffma2_rn(a[i], m, c);
                if (MODE == 1 || MODE == 2) asm volatile("lop3.b32 %0, %0, %1, 0x55555555, 0x96;" : "+r"(u[i]) : "r"(u[(i + 1) & 7]));
                if (MODE == 3) u[i] = __shfl_xor_sync(0xffffffffu, u[i], 1);
                if (MODE == 4) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(sbase + i * 128)); u[i] ^= __float_as_uint(v); }
                if (MODE == 5) a[i] = __fadd2_rn(a[i], c);     // two packed ops
                if (MODE == 6) asm volatile("st.shared.f32 [%0], %1;" :: "r"(sbase + i * 128), "f"(f[i]) : "memory");
                if (MODE == 7) a[i] = __ffma2_rn(a[i], a[(i + 1) & 7], a[(i + 2) & 7]);   // 3 distinct register pairs
                if (MODE == 8) f[i] = fmaf(f[i], 1.0001f, 0.001f);                         // scalar FFMA only
                if (MODE == 9) { f[i] = fmaf(f[i], 1.0001f, 0.001f); asm volatile("lop3.b32 %0, %0, %1, 0x55555555, 0x96;" : "+r"(u[i]) : "r"(u[(i + 1) & 7])); }
                if (MODE == 10) f[i] = fmaf(f[i], 1.0001f, 0.001f);                        // FFMA2 + scalar FFMA
            }
        }
    }
    long long t1 = clock64();
    float s = 0; unsigned x = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { s += a[i].x + a[i].y + f[i]; x ^= u[i]; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s + x;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int M> void run(const char *name, float *out, long long *cyc)
{
    const int iters = 2000; long long h = 0;
    k<M><<<148, 512>>>(out, iters, cyc); cudaDeviceSynchronize(); k<M><<<148, 512>>>(out, iters, cyc);
    cudaError_t e = cudaDeviceSynchronize();
    cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("%-22s %6.2f cycles per slot per SMSP (4 warps/SMSP)  %s\n", name, (double)h / (iters * 32.0) / 4.0, cudaGetErrorString(e));
}
int main()
{
    float *out; long long *cyc;
    cudaMalloc(&out, 148 * 512 * 4); cudaMalloc(&cyc, 8);
    run<0>("FFMA2 only", out, cyc); run<1>("LOP3 only", out, cyc); run<2>("FFMA2+LOP3", out, cyc); run<3>("FFMA2+SHFL", out, cyc);
    run<4>("FFMA2+LDS", out, cyc); run<5>("FFMA2+FADD2", out, cyc); run<6>("FFMA2+STS", out, cyc); run<7>("FFMA2+FFMA2(3reg)", out, cyc);
    run<8>("FFMA only", out, cyc); run<9>("FFMA+LOP3", out, cyc); run<10>("FFMA2+FFMA", out, cyc);
    return 0;
}
