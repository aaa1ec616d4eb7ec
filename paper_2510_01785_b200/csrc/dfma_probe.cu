// Register-operand bandwidth micro-benchmark (a measurement tool outside libcuhpx.so; profiles/r2_dfma_probe.md).
// Question: why do the fp64 Legendre kernels (legendre.cu), whose inner loops are dense DFMA streams with stall
// count 2 on every instruction, stop at 62 % (analysis) and 78 % (synthesis) of the FP64 pipe?
// Part 1 times DFMA streams that differ only in how many source registers are fresh per instruction (not served by
// the operand reuse cache): the pipe issues one warp-DFMA every 2 clk only when at most two 64-bit registers are
// read; a third fresh register costs a third clock.  Part 2 times the inner loops of the two kernels in isolation
// (same arithmetic, nothing else) in the instruction order ptxas chooses.  Part 3 repeats part 1 for FFMA / FFMA2.
// Part 4 runs a DFMA stream and an FFMA2 stream side by side on every sub-partition.
//   build: python -m paper_2510_01785_b200.build --probe        run: ./paper_2510_01785_b200/dfma_probe
#include <cstdio>
#include <cuda_runtime.h>

constexpr double PEAK_TFLOPS = 148 * 64 * 2 * 1.965e-3;  // 148 SM x 64 fp64 FMA lanes x 2 flop x 1.965 GHz

// ---- part 1: 16 independent accumulators, 64 DFMA per loop trip
// T1 acc_k = fma(a, b, acc_k)          one fresh register (acc_k); a and b stay in the reuse cache
// T2 acc_k = fma(a_k, b, acc_k)        two fresh
// T3 acc_k = fma(a_k, b_k, acc_k)      three fresh
// T4 acc_k = fma(a_k, a_k, acc_k)      two distinct registers (a_k read once for both slots)
// T5 acc_k = fma(a_(k/2), b_k, acc_k)  pairs share a: three fresh, then two
template <int T>
__global__ void __launch_bounds__(128, 3) operand_kernel(const double* __restrict__ in, double* __restrict__ out, int n) {
    double a[16], b[16], acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        a[i] = in[i + threadIdx.x];
        b[i] = in[32 + i + threadIdx.x];
        acc[i] = in[64 + i];
    }
#pragma unroll 1
    for (int t = 0; t < n; ++t) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                if (T == 1) acc[i] = fma(a[0], b[0], acc[i]);
                if (T == 2) acc[i] = fma(a[i], b[0], acc[i]);
                if (T == 3) acc[i] = fma(a[i], b[i], acc[i]);
                if (T == 4) acc[i] = fma(a[i], a[i], acc[i]);
                if (T == 5) acc[i] = fma(a[i / 2], b[i], acc[i]);
            }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- part 2: the inner loops of legendre_analysis_kernel<double, 1, R, 8, ...> and legendre_synthesis_kernel<double, 1, R, ...>
// MODE 0 analysis: per degree and ring  acc[2] += lambda * F[2];  lambda <- A (lambda - y lambda) - lambda_prev
// MODE 1 synthesis: per degree and ring  G[ring][parity][2] += lambda * a_lm[2];  same recurrence
// MODE 2 recurrence alone
template <int R, int MODE>
__global__ void __launch_bounds__(64, 6) loop_kernel(const double* __restrict__ in, double* __restrict__ out, int ntiles) {
    __shared__ double sA[64], sRe[64], sIm[64];
    if (threadIdx.x < 64) {
        sA[threadIdx.x] = in[threadIdx.x];
        sRe[threadIdx.x] = in[700 + threadIdx.x];
        sIm[threadIdx.x] = in[800 + threadIdx.x];
    }
    __syncthreads();
    double cur[R], prev[R], y[R], f[R][4], g[R][4];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        cur[r] = in[64 + threadIdx.x + r];
        prev[r] = 0;
        y[r] = in[100 + threadIdx.x + r];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            f[r][c] = in[200 + 100 * c + threadIdx.x + r];
            g[r][c] = 0;
        }
    }
    double tot = 0;
#pragma unroll 1
    for (int t = 0; t < ntiles; ++t) {
        double acc[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int k = (t & 7) * 8 + i;
            const double A = sA[k];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (MODE == 0) {
                    acc[2 * i] = fma(cur[r], f[r][2 * (i & 1)], acc[2 * i]);
                    acc[2 * i + 1] = fma(cur[r], f[r][2 * (i & 1) + 1], acc[2 * i + 1]);
                }
                if (MODE == 1) {
                    g[r][2 * (i & 1)] = fma(cur[r], sRe[k], g[r][2 * (i & 1)]);
                    g[r][2 * (i & 1) + 1] = fma(cur[r], sIm[k], g[r][2 * (i & 1) + 1]);
                }
                const double xl = fma(-y[r], cur[r], cur[r]);
                const double nx = fma(A, xl, -prev[r]);
                prev[r] = cur[r];
                cur[r] = nx;
            }
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) tot += acc[i];
    }
    double s = tot;
#pragma unroll
    for (int r = 0; r < R; ++r) s += cur[r] + g[r][0] + g[r][1] + g[r][2] + g[r][3];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- part 3: the same operand patterns for FFMA and the packed FFMA2 (fma.rn.f32x2) of the fp32 kernels
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}
__device__ __forceinline__ float fmaT(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float2 fmaT(float2 a, float2 b, float2 c) { return fma2(a, b, c); }
__device__ __forceinline__ float sumT(float a) { return a; }
__device__ __forceinline__ float sumT(float2 a) { return a.x + a.y; }

template <typename V, int T>
__global__ void __launch_bounds__(128, 4) operand32_kernel(const V* __restrict__ in, float* __restrict__ out, int n) {
    V a[16], b[16], acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        a[i] = in[i + threadIdx.x];
        b[i] = in[32 + i + threadIdx.x];
        acc[i] = in[64 + i];
    }
#pragma unroll 1
    for (int t = 0; t < n; ++t) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                if (T == 2) acc[i] = fmaT(a[i], b[0], acc[i]);
                if (T == 3) acc[i] = fmaT(a[i], b[i], acc[i]);
                if (T == 4) acc[i] = fmaT(a[i], a[i], acc[i]);
                if (T == 5) acc[i] = fmaT(a[i / 2], b[i], acc[i]);
            }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += sumT(acc[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- part 4: do a DFMA stream and an FFMA2 stream on the SAME sub-partition overlap?  One CTA of 8 warps per SM: warps
// 0-3 (one per sub-partition) run DFMAs, warps 4-7 FFMA2s, each with two fresh operands per instruction (full rate
// alone).  MODE 1: only the DFMA warps work, 2: only the FFMA2 warps, 3: both.
template <int MODE>
__global__ void __launch_bounds__(256, 1) coissue_kernel(const double* __restrict__ in, double* __restrict__ out, int n) {
    const int warp = threadIdx.x >> 5;
    double s = 0;
    if (warp < 4) {
        if (MODE & 1) {
            double a[16], acc[16];
            const double b = in[threadIdx.x];
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                a[i] = in[i + threadIdx.x];
                acc[i] = in[64 + i];
            }
#pragma unroll 1
            for (int t = 0; t < n; ++t)
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int i = 0; i < 16; ++i) acc[i] = fma(a[i], b, acc[i]);
#pragma unroll
            for (int i = 0; i < 16; ++i) s += acc[i];
        }
    } else if (MODE & 2) {
        const float2* fin = reinterpret_cast<const float2*>(in);
        float2 a[16], acc[16];
        const float2 b = fin[threadIdx.x];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            a[i] = fin[i + threadIdx.x];
            acc[i] = fin[64 + i];
        }
#pragma unroll 1
        for (int t = 0; t < n; ++t)
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int i = 0; i < 16; ++i) acc[i] = fma2(a[i], b, acc[i]);
#pragma unroll
        for (int i = 0; i < 16; ++i) s += acc[i].x + acc[i].y;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename K>
static float time_ms(K launch) {
    launch();
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaEventRecord(e0);
    launch();
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    return ms;
}

template <int T>
static void run_operand(const char* what, const double* in, double* out) {
    const int n = 4000, grid = 148 * 12;
    const float ms = time_ms([&] { operand_kernel<T><<<grid, 128>>>(in, out, n); });
    const double tf = 2.0 * 64 * n * (double)grid * 128 / ms * 1e-9;
    printf("%-44s %6.2f TFLOP/s  %5.1f %% of the FP64 pipe  -> %.2f clk per warp-DFMA\n", what, tf, 100 * tf / PEAK_TFLOPS,
           2.0 * PEAK_TFLOPS / tf);
}

template <int R, int MODE>
static void run_loop(const char* what, const double* in, double* out) {
    const int ntiles = 2000, grid = 148 * 24;
    const float ms = time_ms([&] { loop_kernel<R, MODE><<<grid, 64>>>(in, out, ntiles); });
    const double per_tile = (MODE == 2 ? 2.0 : 4.0) * R * 8 + (MODE == 0 ? 16 : 0);  // DFMA + the 16 DADD of the tile sums
    const double tf = 2.0 * per_tile * ntiles * (double)grid * 64 / ms * 1e-9;
    printf("%-44s %6.2f TFLOP/s  %5.1f %% of the FP64 pipe  -> %.2f clk per warp-DFMA\n", what, tf, 100 * tf / PEAK_TFLOPS,
           2.0 * PEAK_TFLOPS / tf);
}

template <typename V, int T>
static void run_operand32(const char* what, const double* in, double* out) {
    const int n = 8000, grid = 148 * 16;
    const float ms = time_ms([&] { operand32_kernel<V, T><<<grid, 128>>>(reinterpret_cast<const V*>(in), reinterpret_cast<float*>(out), n); });
    const double lanes = sizeof(V) / 4;  // FMAs per lane and instruction
    const double tf = 2.0 * lanes * 64 * n * (double)grid * 128 / ms * 1e-9;
    printf("%-44s %6.2f TFLOP/s  %5.1f %% of the FMA pipe   -> %.2f clk per warp-instruction\n", what, tf, 100 * tf / (2 * PEAK_TFLOPS),
           lanes * 2.0 * PEAK_TFLOPS / tf);
}

int main() {
    double *in, *out;
    cudaMalloc(&in, 8192);
    cudaMemset(in, 0, 8192);
    cudaMalloc(&out, sizeof(double) * 148 * 24 * 128);
    printf("FP64 pipe peak used below: %.1f TFLOP/s (148 SM x 64 lanes x 2 x 1.965 GHz); 3 warps per SM sub-partition\n", PEAK_TFLOPS);
    printf("-- part 1: fresh source registers per DFMA\n");
    run_operand<1>("T1 fma(a, b, acc_k)         1 fresh", in, out);
    run_operand<2>("T2 fma(a_k, b, acc_k)       2 fresh", in, out);
    run_operand<4>("T4 fma(a_k, a_k, acc_k)     2 distinct", in, out);
    run_operand<5>("T5 fma(a_(k/2), b_k, acc_k) 3 then 2 fresh", in, out);
    run_operand<3>("T3 fma(a_k, b_k, acc_k)     3 fresh", in, out);
    printf("-- part 2: the Legendre inner loops alone, ptxas instruction order\n");
    run_loop<7, 2>("recurrence only, 7 ring pairs", in, out);
    run_loop<7, 0>("analysis loop, 7 ring pairs, 8 degrees", in, out);
    run_loop<6, 0>("analysis loop, 6 ring pairs, 8 degrees", in, out);
    run_loop<6, 1>("synthesis loop, 6 ring pairs", in, out);
    run_loop<4, 1>("synthesis loop, 4 ring pairs", in, out);
    printf("-- part 3: FFMA / FFMA2 (fp32 peak %.1f TFLOP/s: one FFMA per clk, one FFMA2 per 2 clk and sub-partition)\n", 2 * PEAK_TFLOPS);
    run_operand32<float, 2>("FFMA  fma(a_k, b, acc_k)       2 fresh", in, out);
    run_operand32<float, 5>("FFMA  fma(a_(k/2), b_k, acc_k) 3 then 2 fresh", in, out);
    run_operand32<float, 3>("FFMA  fma(a_k, b_k, acc_k)     3 fresh", in, out);
    run_operand32<float2, 2>("FFMA2 fma(a_k, b, acc_k)       2 fresh pairs", in, out);
    run_operand32<float2, 4>("FFMA2 fma(a_k, a_k, acc_k)     2 distinct pairs", in, out);
    run_operand32<float2, 5>("FFMA2 fma(a_(k/2), b_k, acc_k) 3 then 2 fresh", in, out);
    run_operand32<float2, 3>("FFMA2 fma(a_k, b_k, acc_k)     3 fresh pairs", in, out);
    printf("-- part 4: one DFMA warp and one FFMA2 warp per sub-partition (64 instructions x 20000 trips per warp)\n");
    {
        const int n = 20000;
        const float t1 = time_ms([&] { coissue_kernel<1><<<148, 256>>>(in, out, n); });
        const float t2 = time_ms([&] { coissue_kernel<2><<<148, 256>>>(in, out, n); });
        const float t3 = time_ms([&] { coissue_kernel<3><<<148, 256>>>(in, out, n); });
        const double clk = 1.965e6;  // clocks per ms
        printf("DFMA warps alone  %.3f ms = %.2f clk per DFMA\n", t1, t1 * clk / (64.0 * n));
        printf("FFMA2 warps alone %.3f ms = %.2f clk per FFMA2\n", t2, t2 * clk / (64.0 * n));
        printf("both together     %.3f ms  (sum %.3f, max %.3f)\n", t3, t1 + t2, t1 > t2 ? t1 : t2);
    }
    const cudaError_t e = cudaDeviceSynchronize();
    printf("%s\n", cudaGetErrorString(e));
    return e != cudaSuccess;
}
