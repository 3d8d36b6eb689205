// microbenchmarks behind DESIGN.md 7.1 (lower-bound model of the batch-1 step): pipe throughputs (per SM, clocks per warp-instruction),
// L2-hit latency of ld.relaxed.gpu, store -> poll hop between two CTAs, cost of fence.acq_rel.gpu.  Build and run:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -fmad=false -o /tmp/hop_ubench paper_2606_10932_b200/bench_micro/hop_ubench.cu && /tmp/hop_ubench
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

template <int OP>
__global__ void k_tput(int iters, int* out, long long* clk)
{
    int a0 = threadIdx.x, a1 = a0 * 3 + 1, a2 = a0 ^ 0x55, a3 = a0 + 7, a4 = a0 * 5, a5 = a0 + 11, a6 = a0 * 7, a7 = a0 ^ 99;
    int b = blockIdx.x + 0x01020304;
    double d0 = a0, d1 = a1, d2 = a2, d3 = a3;
    float f0 = a0, f1 = a1, f2 = a2, f3 = a3;
    __syncthreads();
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
        if (OP == 0) {   // dp4a u8.s8 x8 independent chains
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a0) : "r"(b), "r"(a1));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a2) : "r"(b), "r"(a3));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a4) : "r"(b), "r"(a5));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a6) : "r"(b), "r"(a7));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a1) : "r"(b), "r"(a0));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a3) : "r"(b), "r"(a2));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a5) : "r"(b), "r"(a4));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a7) : "r"(b), "r"(a6));
        } else if (OP == 1) {   // lop3 x8
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a0) : "r"(b), "r"(a1));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a2) : "r"(b), "r"(a3));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a4) : "r"(b), "r"(a5));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a6) : "r"(b), "r"(a7));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a1) : "r"(b), "r"(a0));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a3) : "r"(b), "r"(a2));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a5) : "r"(b), "r"(a4));
            asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a7) : "r"(b), "r"(a6));
        } else if (OP == 2) {   // 4 x (lop3 + dp4a)
            int m0, m1, m2, m3;
            asm volatile("and.b32 %0, %1, 0x01010101;" : "=r"(m0) : "r"(b));
            asm volatile("and.b32 %0, %1, 0x02020202;" : "=r"(m1) : "r"(b));
            asm volatile("and.b32 %0, %1, 0x04040404;" : "=r"(m2) : "r"(b));
            asm volatile("and.b32 %0, %1, 0x08080808;" : "=r"(m3) : "r"(b));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a0) : "r"(m0), "r"(a1));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a2) : "r"(m1), "r"(a3));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a4) : "r"(m2), "r"(a5));
            asm volatile("dp4a.u32.s32 %0, %1, %2, %0;" : "+r"(a6) : "r"(m3), "r"(a7));
            b += a0 & 1;
        } else if (OP == 3) {   // cvt f32 -> f64 x4 + dfma x4
            d0 = __fma_rn((double)f0, d1, d0); d1 = __fma_rn((double)f1, d2, d1);
            d2 = __fma_rn((double)f2, d3, d2); d3 = __fma_rn((double)f3, d0, d3);
            f0 += 1.0f; f1 += 1.0f; f2 += 1.0f; f3 += 1.0f;
        } else if (OP == 4) {   // dfma x8 only
            d0 = __fma_rn(d0, d1, d2); d1 = __fma_rn(d1, d2, d3); d2 = __fma_rn(d2, d3, d0); d3 = __fma_rn(d3, d0, d1);
            d0 = __fma_rn(d0, d1, d2); d1 = __fma_rn(d1, d2, d3); d2 = __fma_rn(d2, d3, d0); d3 = __fma_rn(d3, d0, d1);
        } else if (OP == 5) {   // i2f.f64 x4 + dadd
            d0 += (double)a0; d1 += (double)a1; d2 += (double)a2; d3 += (double)a3;
            a0 += 3; a1 += 5; a2 += 7; a3 += 9;
        } else if (OP == 6) {   // imad x8
            a0 = a0 * b + a1; a2 = a2 * b + a3; a4 = a4 * b + a5; a6 = a6 * b + a7;
            a1 = a1 * b + a0; a3 = a3 * b + a2; a5 = a5 * b + a4; a7 = a7 * b + a6;
        } else if (OP == 7) {   // ffma x8
            f0 = __fmaf_rn(f0, f1, f2); f1 = __fmaf_rn(f1, f2, f3); f2 = __fmaf_rn(f2, f3, f0); f3 = __fmaf_rn(f3, f0, f1);
            f0 = __fmaf_rn(f0, f1, f2); f1 = __fmaf_rn(f1, f2, f3); f2 = __fmaf_rn(f2, f3, f0); f3 = __fmaf_rn(f3, f0, f1);
        }
    }
    long long t1 = clock64();
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7 + (int)(d0 + d1 + d2 + d3) + (int)(f0 + f1 + f2 + f3);
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// latency of one ld.relaxed.gpu (L2 hit) chain, and of a store -> remote poll hop between 2 CTAs
__global__ void k_l2lat(uint32_t* buf, int n, long long* clk)
{
    if (threadIdx.x != 0) return;
    uint32_t idx = 0;
    long long t0 = clock64();
    for (int i = 0; i < n; ++i) {
        uint32_t v;
        asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(buf + idx) : "memory");
        idx = v;
    }
    long long t1 = clock64();
    clk[blockIdx.x] = (t1 - t0) / n + (idx == 12345);
}
// ping-pong between CTA 0 and CTA `peer`: round trip = 2 hops
__global__ void k_pingpong(volatile uint32_t* flags, int peer, int rounds, long long* clk)
{
    if (threadIdx.x != 0) return;
    const int me = blockIdx.x;
    if (me != 0 && me != peer) return;
    uint32_t* mine = (uint32_t*)flags + (me == 0 ? 0 : 64), *other = (uint32_t*)flags + (me == 0 ? 64 : 0);
    long long t0 = clock64();
    for (int r = 1; r <= rounds; ++r) {
        if (me == 0) {
            asm volatile("st.relaxed.gpu.global.b32 [%0], %1;" ::"l"(other), "r"(r) : "memory");
            uint32_t v;
            do { asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(mine) : "memory"); } while (v != (uint32_t)r);
        } else {
            uint32_t v;
            do { asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(mine) : "memory"); } while (v != (uint32_t)r);
            asm volatile("st.relaxed.gpu.global.b32 [%0], %1;" ::"l"(other), "r"(r) : "memory");
        }
    }
    long long t1 = clock64();
    if (me == 0) clk[0] = (t1 - t0) / rounds;
}
// fence cost: one thread, fence.acq_rel.gpu with no outstanding stores / after one store
__global__ void k_fence(uint32_t* buf, int n, long long* clk)
{
    if (threadIdx.x != 0) return;
    long long t0 = clock64();
    for (int i = 0; i < n; ++i) asm volatile("fence.acq_rel.gpu;" ::: "memory");
    long long t1 = clock64();
    for (int i = 0; i < n; ++i) { asm volatile("st.relaxed.gpu.global.b32 [%0], %1;" ::"l"(buf + blockIdx.x * 32), "r"(i) : "memory"); asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
    long long t2 = clock64();
    clk[2 * blockIdx.x] = (t1 - t0) / n; clk[2 * blockIdx.x + 1] = (t2 - t1) / n;
}

int main()
{
    int* out; long long* clk; uint32_t* buf;
    CK(cudaMalloc(&out, 148 * 1024 * 4)); CK(cudaMalloc(&clk, 148 * 16 * 8)); CK(cudaMalloc(&buf, 1 << 24));
    long long h[148 * 2];
    const int iters = 4096;
    const char* names[] = { "dp4a x8", "lop3 x8", "4x(and+dp4a)", "4x(cvt f32->f64 + dfma)", "dfma x8", "4x(i2f.f64+dadd)", "imad x8", "ffma x8" };
    const int nin[] = { 8, 8, 9, 12, 8, 12, 8, 8 };
    for (int nw = 4; nw <= 16; nw *= 2) {
        printf("-- %d warps per SM (1 CTA/SM), clocks per warp-instruction per SM (ideal 0.25 = 4 IPC)\n", nw);
#define RUN(OP) { k_tput<OP><<<148, nw * 32>>>(iters, out, clk); CK(cudaDeviceSynchronize()); CK(cudaMemcpy(h, clk, 8, cudaMemcpyDeviceToHost)); \
        printf("   %-26s %7.3f clk per warp-instr/SM  (%.2f clk per loop iter per warp)\n", names[OP], (double)h[0] / iters / nin[OP] / nw, (double)h[0] / iters); }
        RUN(0) RUN(1) RUN(2) RUN(3) RUN(4) RUN(5) RUN(6) RUN(7)
    }
    // L2 latency: pointer chase within 1 MB (L2 resident), stride 4 KB+
    {
        const int N = 4096; static uint32_t hb[1 << 20];
        for (int i = 0; i < (1 << 20); ++i) hb[i] = 0;
        uint32_t idx = 0;
        for (int i = 0; i < N; ++i) { uint32_t nx = (uint32_t)(((long long)(i + 1) * 7919 * 64) % (1 << 20)); hb[idx] = nx; idx = nx; }
        CK(cudaMemcpy(buf, hb, sizeof hb, cudaMemcpyHostToDevice));
        k_l2lat<<<148, 32>>>(buf, 2000, clk); CK(cudaDeviceSynchronize());
        k_l2lat<<<148, 32>>>(buf, 2000, clk); CK(cudaDeviceSynchronize());
        CK(cudaMemcpy(h, clk, 148 * 8, cudaMemcpyDeviceToHost));
        long long mn = 1 << 30, mx = 0, s = 0; for (int i = 0; i < 148; ++i) { mn = h[i] < mn ? h[i] : mn; mx = h[i] > mx ? h[i] : mx; s += h[i]; }
        printf("ld.relaxed.gpu L2-hit latency (148 CTAs chasing): min %lld mean %lld max %lld clocks\n", mn, s / 148, mx);
        k_l2lat<<<1, 32>>>(buf, 2000, clk); CK(cudaDeviceSynchronize());
        CK(cudaMemcpy(h, clk, 8, cudaMemcpyDeviceToHost));
        printf("ld.relaxed.gpu L2-hit latency (1 CTA): %lld clocks\n", h[0]);
    }
    for (int peer : { 1, 2, 37, 74, 100, 147 }) {
        CK(cudaMemset(buf, 0, 1024));
        void* args[] = { &buf, &peer, (void*)&iters, &clk };
        int rounds = 2000; args[2] = &rounds;
        CK(cudaLaunchCooperativeKernel((void*)k_pingpong, dim3(148), dim3(32), args, 0, 0)); CK(cudaDeviceSynchronize());
        CK(cudaMemcpy(h, clk, 8, cudaMemcpyDeviceToHost));
        printf("ping-pong CTA0 <-> CTA%d: round trip %lld clocks (one hop = %lld)\n", peer, h[0], h[0] / 2);
    }
    k_fence<<<1, 32>>>(buf, 1000, clk); CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(h, clk, 16, cudaMemcpyDeviceToHost));
    printf("fence.acq_rel.gpu: %lld clocks idle, %lld clocks after one store\n", h[0], h[1]);
    return 0;
}
