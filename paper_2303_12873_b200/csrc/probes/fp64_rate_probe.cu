// fp64_rate_probe.cu -- cycles per warp instruction per SM of DFMA and DMMA (m8n8k4, m16n8k8), one block per SM.
// Not part of the library: it backs the fp64-pipe peak DESIGN.md 5 derives (64 lanes/clk/SM).
// nvcc -gencode arch=compute_100a,code=sm_100a -O2 -o fp64_rate_probe fp64_rate_probe.cu && ./fp64_rate_probe
#include <cstdio>
#include <cuda_runtime.h>
__global__ void probe(int mode, int iters, long long* out, double* sink) {
    double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-4;
    double c[8][2];
    for (int k = 0; k < 8; ++k) c[k][0] = c[k][1] = 0.0;
    __syncthreads();
    long long t0 = clock64();
    if (mode == 0) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
        }
    } else if (mode == 1) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(c[k][0]) : "d"(a), "d"(b));
                asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(c[k][1]) : "d"(a), "d"(b));
            }
        }
    } else {
        // m16n8k8: A 4 regs, B 2 regs, C 4 regs
        double c4[4][4];
        for (int k = 0; k < 4; ++k) for (int j = 0; j < 4; ++j) c4[k][j] = 0.0;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                             : "+d"(c4[k][0]), "+d"(c4[k][1]), "+d"(c4[k][2]), "+d"(c4[k][3])
                             : "d"(a), "d"(b), "d"(a), "d"(b), "d"(a), "d"(b));
        }
        for (int k = 0; k < 4; ++k) for (int j = 0; j < 4; ++j) c[k][j & 1] += c4[k][j];
    }
    long long t1 = clock64();
    double s = 0;
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    if (s == 12345.678) sink[0] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) out[0] = t1 - t0;
}
int main() {
    long long* out; double* sink;
    cudaMalloc(&out, 8); cudaMalloc(&sink, 8);
    int iters = 2000;
    for (int warps : {4, 8, 16}) {
        for (int mode = 0; mode < 3; ++mode) {
            probe<<<148, warps * 32>>>(mode, iters, out, sink);
            long long h; cudaMemcpy(&h, out, 8, cudaMemcpyDeviceToHost);
            const char* nm = mode == 0 ? "DMMA m8n8k4 (256 FMA)" : (mode == 1 ? "DFMA x2 (64 FMA)" : "DMMA m16n8k8 (1024 FMA)");
            double per = mode == 2 ? (double)h / (iters * 4.0 * warps) : (double)h / (iters * 8.0 * warps);
            printf("warps %2d  %-28s %.2f clk per warp-instr(group) per SM\n", warps, nm, per);
        }
    }
    return 0;
}
