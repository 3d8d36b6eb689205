// instruction-fetch cost: a straight-line body of N distinct FFMA-chains (4 independent chains) executed in a loop by 16 warps/SM
#include <cstdio>
#include <cuda_runtime.h>
#define R4(k)  a0 = a0 * 1.0001f + (k + 0.1f); a1 = a1 * 1.0002f + (k + 0.2f); a2 = a2 * 1.0003f + (k + 0.3f); a3 = a3 * 1.0004f + (k + 0.4f);
#define R16(k) R4(k) R4(k + 1) R4(k + 2) R4(k + 3)
#define R64(k) R16(k) R16(k + 4) R16(k + 8) R16(k + 12)
#define R256(k) R64(k) R64(k + 16) R64(k + 32) R64(k + 48)
#define R1K(k) R256(k) R256(k + 64) R256(k + 128) R256(k + 192)
template <int KB>   // body of KB * 1024 / 16 instructions
__global__ void k(int iters, float* out, long long* clk)
{
    float a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3;
    __syncthreads();
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
        // each R4 = 4 FFMA = 64 bytes; R1K = 1024 FFMA... R256(k) = 256*... careful: R4 has 4 instr, R16 16, R64 64, R256 256, R1K 1024 instrs = 16 KB
        if (KB >= 16) { R1K(0) }
        if (KB >= 32) { R1K(1000) }
        if (KB >= 48) { R1K(2000) }
        if (KB >= 64) { R1K(3000) }
        if (KB >= 96) { R1K(4000) R1K(5000) }
        if (KB >= 128) { R1K(6000) R1K(7000) }
        if (KB == 4) { R256(0) }
        if (KB == 8) { R256(0) R256(300) }
        __syncthreads();
    }
    long long t1 = clock64();
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}
template <int KB> void run(int nw, float* out, long long* clk)
{
    const int iters = 200;
    k<KB><<<148, nw * 32>>>(iters, out, clk); cudaDeviceSynchronize();
    k<KB><<<148, nw * 32>>>(iters, out, clk); cudaDeviceSynchronize();
    long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
    const double ninstr = KB * 1024.0 / 16.0;
    printf("body %3d KB, %2d warps: %8.1f clocks per pass, %.2f clocks per instruction per warp, SM IPC %.2f\n", KB, nw, (double)h / iters,
           (double)h / iters / ninstr, ninstr * nw / ((double)h / iters));
}
int main()
{
    float* out; long long* clk; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&clk, 148 * 8);
    for (int nw : { 1, 4, 16 }) {
        run<4>(nw, out, clk); run<8>(nw, out, clk); run<16>(nw, out, clk); run<32>(nw, out, clk); run<48>(nw, out, clk); run<64>(nw, out, clk);
        run<96>(nw, out, clk); run<128>(nw, out, clk);
    }
    return 0;
}
