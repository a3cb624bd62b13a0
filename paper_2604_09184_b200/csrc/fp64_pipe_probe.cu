// fp64_pipe_probe.cu -- standalone measurement aid (not part of libnbkick.so): what the B200 FP64 pipe
// really sustains for the operand patterns and instruction mixes of the force-tile kernel.
//   build:  python -m paper_2604_09184_b200.build --probe      run:  paper_2604_09184_b200/fp64_pipe_probe
// Every operand is thread-dependent, so it lives in vector registers (uniform-register operands do not
// load the register-file read ports and would hide the effect).  Results: profiles/r1_fp64_pipe_microbench.md
#include <cstdio>
#include <cuda_runtime.h>

template <int P>
__global__ void __launch_bounds__(256) operand_kernel(double *out, int iters, const double *src) {
    double c[8], p[8], q[8], s[3];
    const double tid = threadIdx.x * 1e-9;
    for (int r = 0; r < 8; ++r) { c[r] = tid + r; p[r] = src[r] + tid; q[r] = src[8 + r] - tid; }
    for (int r = 0; r < 3; ++r) s[r] = src[r] * tid;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (P == 1) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __dadd_rn(c[r], p[r]); }
            if (P == 2) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __dmul_rn(c[r], p[r]); }
            if (P == 3) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __fma_rn(c[r], p[r], q[r]); }
            if (P == 4) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __fma_rn(p[r], p[r], c[r]); }
            if (P == 5) {  // accumulate triplets sharing s, adjacent (operand-reuse-cache friendly)
                c[0] = __fma_rn(s[0], p[0], c[0]); c[1] = __fma_rn(s[0], p[1], c[1]); c[2] = __fma_rn(s[0], p[2], c[2]);
                c[3] = __fma_rn(s[1], p[3], c[3]); c[4] = __fma_rn(s[1], p[4], c[4]); c[5] = __fma_rn(s[1], p[5], c[5]);
                c[6] = __fma_rn(s[2], p[6], c[6]); c[7] = __fma_rn(s[2], p[7], c[7]);
            }
            if (P == 6) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __fma_rn(c[r], p[r], 1.0); }
            if (P == 7) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __fma_rn(c[r], p[0], q[0]); }
            if (P == 8) { _Pragma("unroll") for (int r = 0; r < 8; ++r) c[r] = __fma_rn(p[r], q[r], c[r]); }
        }
    }
    double t = 0;
    for (int r = 0; r < 8; ++r) t += c[r];
    if (t == 123.456) out[0] = t;
}

// 8 two-read DFMAs (2 clk each) + NI instructions of another pipe per group
template <int NI, int KIND>
__global__ void __launch_bounds__(256) mix_kernel(double *out, int iters, const double *src, int seed) {
    double c[8], p[8], l[8];
    int z[8];
    float f[8];
    const double tid = threadIdx.x * 1e-9;
    for (int r = 0; r < 8; ++r) {
        c[r] = tid + r; p[r] = src[r] + tid; z[r] = seed + r + threadIdx.x; f[r] = seed * 0.5f + r + threadIdx.x; l[r] = 0;
    }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                c[r] = __fma_rn(p[r], p[r], c[r]);
                if (r < NI) {
                    if (KIND == 1) f[r] = fmaf(f[r], 0.99f, 1.5f);  // FFMA
                    if (KIND == 2) z[r] = max(z[r], seed + u);      // VIMNMX
                    if (KIND == 3) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(c[r])); l[r] = y; }  // MUFU.RSQ64H (+MOV)
                }
            }
        }
    }
    double s = 0;
    for (int r = 0; r < 8; ++r) s += c[r] + z[r] + f[r] + l[r];
    if (s == 123.456) out[0] = s;
}

static double *g_d, *g_src;
static cudaEvent_t g_e0, g_e1;
static const int kIters = 2048, kCtas = 148 * 4;

template <typename F>
static void time_it(const char *name, F launch) {
    float ms = 1e9f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(g_e0);
        launch();
        cudaEventRecord(g_e1);
        cudaEventSynchronize(g_e1);
        float t;
        cudaEventElapsedTime(&t, g_e0, g_e1);
        if (t < ms) ms = t;
    }
    const double inst = (double)kCtas * 256 * kIters * 64.0;  // fp64 thread-instructions
    printf("%-52s %7.3f ms   fp64 issue rate = %5.1f%% of 1 warp-instr / 2 clk / SMSP @1.965 GHz\n", name, ms,
           100.0 * inst / (ms * 1e-3) / (148.0 * 64 * 1.965e9));
}
#define OP(P, name) time_it(name, [] { operand_kernel<P><<<kCtas, 256>>>(g_d, kIters, g_src); })
#define MIX(NI, KIND, name) time_it(name, [] { mix_kernel<NI, KIND><<<kCtas, 256>>>(g_d, kIters, g_src, 3); })

int main() {
    cudaMalloc(&g_d, 256); cudaMalloc(&g_src, 256); cudaMemset(g_src, 0, 256);
    cudaEventCreate(&g_e0); cudaEventCreate(&g_e1);
    OP(1, "(warm-up)"); OP(1, "(warm-up)");
    OP(1, "DADD  c = c + p            (2 register pairs read)");
    OP(2, "DMUL  c = c * p            (2 pairs)");
    OP(4, "DFMA  c = p*p + c          (2 distinct pairs)");
    OP(6, "DFMA  c = c*p + 1.0        (2 pairs + immediate)");
    OP(3, "DFMA  c = c*p + q          (3 distinct pairs)");
    OP(8, "DFMA  c = p*q + c          (3 distinct pairs, accumulate)");
    OP(5, "DFMA  c_k = s*p_k + c_k    (s shared by 3 adjacent)");
    OP(7, "DFMA  c = c*p0 + q0        (p0,q0 shared by all 8)");
    MIX(0, 0, "8 DFMA(2-read)");
    MIX(2, 2, "8 DFMA + 2 VIMNMX"); MIX(4, 2, "8 DFMA + 4 VIMNMX"); MIX(8, 2, "8 DFMA + 8 VIMNMX");
    MIX(2, 1, "8 DFMA + 2 FFMA"); MIX(4, 1, "8 DFMA + 4 FFMA"); MIX(8, 1, "8 DFMA + 8 FFMA");
    MIX(1, 3, "8 DFMA + 1 MUFU.RSQ64H"); MIX(2, 3, "8 DFMA + 2 MUFU.RSQ64H"); MIX(4, 3, "8 DFMA + 4 MUFU.RSQ64H");
    return 0;
}
