// p3t_pipebench.cu -- micro-benchmarks of the FP32 pipe of the device the library runs on: the
// per-instruction pipe costs that DESIGN.md section 6 uses to derive the ALU roofline of k_force
// (the driver's MEASURED_PEAKS.json holds HBM and bf16 tensor peaks, no FP32 figure).
// Eight independent chains per thread, 2 CTAs of 256 threads per SM, CUDA events; a result is the
// number of SM-clock cycles one warp instruction (or instruction group) occupies an SM sub-partition.
// Built into its own library, libp3t_diag.so (include/p3t_diag.h): diagnostics, not part of libp3t.so.
// `python -m paper_2110_11658_b200.pipebench` prints the table.
#include <cuda_runtime.h>
#include "p3t_diag.h"
#include "p3t_f32x2.cuh"

__device__ __forceinline__ f2 vfma2(f2 a, f2 b, f2 c) { f2 r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f2 vmul2(f2 a, f2 b) { f2 r; asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ float vfma1(float a, float b, float c) { float r; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }
__device__ __forceinline__ float vrsq(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// MODE 0: FFMA, operands in the reuse cache        1: FFMA2, two distinct register pairs (a, a, c)
//      2: FFMA2, three distinct register pairs     3: FMUL2
//      4: FMUL2 + FFMA alternating (per pair)      5: 8 FMUL2 + 2 MUFU.RSQ (per group of 10)
//      6: MUFU.RSQ alone                            7: FFMA, three distinct registers (bank conflicts as allocated)
//      8: FFMA2, three distinct register pairs of which one is the SAME in consecutive instructions (what two targets per
//         lane would give the p-c loop: q . d_A, q . d_B share the cell operand, so the reuse cache can serve it)
template <int MODE> __global__ void __launch_bounds__(256) k_pipe(float* out, int iters, float s)
{
    f2 a[8], b[8], c[8]; float t[8], u[8], v[8];
    for (int i = 0; i < 8; ++i) {
        a[i] = pk(threadIdx.x * 0.001f + i, 1.0f + i); b[i] = pk(0.5f + i * s, s); c[i] = pk((float)i, s * i);
        t[i] = s * i + threadIdx.x; u[i] = s + i; v[i] = 1.0f + i * s;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE == 0) t[i] = vfma1(t[i], s, s);
            if (MODE == 7) t[i] = vfma1(u[i], v[i], t[i]);
            if (MODE == 1) c[i] = vfma2(a[i], a[i], c[i]);
            if (MODE == 2) c[i] = vfma2(a[i], b[i], c[i]);
            if (MODE == 8) c[i] = vfma2(a[i], b[0], c[i]);
            if (MODE == 3) c[i] = vmul2(c[i], b[i]);
            if (MODE == 4) { c[i] = vmul2(c[i], b[i]); t[i] = vfma1(t[i], s, s); }
            if (MODE == 5) { c[i] = vmul2(c[i], b[i]); if ((i & 3) == 0) t[i] = vrsq(t[i]); }
            if (MODE == 6) t[i] = vrsq(t[i]);
        }
    }
    float r = 0;
    for (int i = 0; i < 8; ++i) r += f2lo(c[i]) + f2hi(c[i]) + t[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

template <int MODE> static float time_mode(float* d, int blocks, int iters, cudaEvent_t e0, cudaEvent_t e1)
{
    float ms = 0;
    for (int rep = 0; rep < 2; ++rep) {                         // the second run is timed
        cudaEventRecord(e0);
        k_pipe<MODE><<<blocks, 256>>>(d, iters, 1.0001f);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
    }
    return ms;
}

extern "C" int p3t_diag_pipe_bench(int device, double* cycles_out, int n_out, double* sm_clock_mhz, int* num_sms)
{
    if (!cycles_out || n_out < 8) return -1;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { (void)cudaGetLastError(); return -1; }
    cudaSetDevice(device);
    int sms = 0, khz = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, device);
    const int bps = 2, iters = 20000, blocks = sms * bps;
    float* d = nullptr;
    if (cudaMalloc(&d, (size_t)blocks * 256 * sizeof(float)) != cudaSuccess) { (void)cudaGetLastError(); return -3; }
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int w = 0; w < 40; ++w) (void)time_mode<3>(d, blocks, iters, e0, e1);     // ~50 ms of load: let the SM clock settle
    float ms[8];
    ms[0] = time_mode<0>(d, blocks, iters, e0, e1); ms[1] = time_mode<1>(d, blocks, iters, e0, e1);
    ms[2] = time_mode<2>(d, blocks, iters, e0, e1); ms[3] = time_mode<3>(d, blocks, iters, e0, e1);
    ms[4] = time_mode<4>(d, blocks, iters, e0, e1); ms[5] = time_mode<5>(d, blocks, iters, e0, e1);
    ms[6] = time_mode<6>(d, blocks, iters, e0, e1); ms[7] = time_mode<7>(d, blocks, iters, e0, e1);
    const float ms8 = time_mode<8>(d, blocks, iters, e0, e1);
    // per SM sub-partition: bps * 8 warps / 4 sub-partitions = 4 warps, each 8 instruction groups per iteration
    const double groups = (double)iters * 8.0 * (bps * 2);
    for (int k = 0; k < 8; ++k) cycles_out[k] = (double)ms[k] * 1e-3 * (double)khz * 1e3 / groups;
    cycles_out[5] *= 8.0;                                       // mode 5: cycles per group of 8 FMUL2 + 2 MUFU.RSQ
    if (n_out >= 9) cycles_out[8] = (double)ms8 * 1e-3 * (double)khz * 1e3 / groups;
    if (sm_clock_mhz) *sm_clock_mhz = khz * 1e-3;
    if (num_sms) *num_sms = sms;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}
