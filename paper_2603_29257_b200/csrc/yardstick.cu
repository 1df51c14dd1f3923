// yardstick.cu -- FP64 arithmetic yardsticks measured on the device itself (include/risp_debug.h, risp_debug_yardstick).
//
// The roofline fractions of bench.py need denominators that MEASURED_PEAKS.json does not carry: the FP64 ALU (DFMA) rate the
// integral passes (Eq. 14, 16) are bound by, and the issue rate of DMMA.8x8x4, the only FP64 tensor
// instruction of sm_100a, which bounds every dense contraction (Eq. 12, 17, 22, 23).  Both kernels keep all operands in
// registers and run long independent dependency chains on every SM sub-partition, so they measure the pipes, nothing else.
#include "ctx.h"

namespace {

constexpr int YS_CHAINS = 16, YS_ITERS = 2048;

__global__ void __launch_bounds__(256) dfma_chain_kernel(double *out, double a, double b)
{
    double acc[YS_CHAINS];
#pragma unroll
    for (int c = 0; c < YS_CHAINS; ++c) acc[c] = (double)(threadIdx.x + c);
    for (int it = 0; it < YS_ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < YS_CHAINS; ++c) acc[c] = fma(acc[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < YS_CHAINS; ++c) s += acc[c];
    if (s == 123.456) out[0] = s;            // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) dmma_chain_kernel(double *out, double a, double b)
{
    double acc[YS_CHAINS][2];
#pragma unroll
    for (int c = 0; c < YS_CHAINS; ++c) { acc[c][0] = (double)threadIdx.x; acc[c][1] = (double)c; }
    for (int it = 0; it < YS_ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < YS_CHAINS; ++c)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(acc[c][0]), "+d"(acc[c][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < YS_CHAINS; ++c) s += acc[c][0] + acc[c][1];
    if (s == 123.456) out[0] = s;
}

}  // namespace

extern "C" int risp_debug_yardstick(risp_ctx *ctx, int which, size_t bytes, int reps, double *out)
{
    if (!out || reps <= 0 || which < 0 || which > 2) return RISP_EINVAL;
    RISP_CUDA_TRY(cudaSetDevice(ctx ? ctx->device : 0));
    int dev = 0, sms = 0;
    RISP_CUDA_TRY(cudaGetDevice(&dev));
    RISP_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    DevScratch scr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    RISP_CUDA_TRY(cudaEventCreate(&e0));
    RISP_CUDA_TRY(cudaEventCreate(&e1));
    float ms = 0.f;
    double work = 0.0;
    cudaError_t err = cudaSuccess;
    if (which == 2) {
        if (bytes < 2) bytes = (size_t)1 << 30;
        char *a = nullptr, *b = nullptr;
        if ((err = scr.alloc(a, bytes)) == cudaSuccess && (err = scr.alloc(b, bytes)) == cudaSuccess) {
            cudaMemsetAsync(a, 1, bytes, 0);
            cudaMemcpyAsync(b, a, bytes, cudaMemcpyDeviceToDevice, 0);
            cudaEventRecord(e0, 0);
            for (int r = 0; r < reps; ++r) cudaMemcpyAsync(b, a, bytes, cudaMemcpyDeviceToDevice, 0);
            cudaEventRecord(e1, 0);
            err = cudaEventSynchronize(e1);
            work = 2.0 * (double)bytes * reps;
        }
    } else {
        double *o = nullptr;
        if ((err = scr.alloc(o, 1)) == cudaSuccess) {
            const int grid = sms * 8;        // 8 CTAs of 8 warps per SM: 16 warps per sub-partition
            auto launch = [&]() {
                if (which == 0) dfma_chain_kernel<<<grid, 256>>>(o, 0.999999, 1e-9);
                else dmma_chain_kernel<<<grid, 256>>>(o, 0.999999, 1e-9);
            };
            launch();
            cudaEventRecord(e0, 0);
            for (int r = 0; r < reps; ++r) launch();
            cudaEventRecord(e1, 0);
            err = cudaEventSynchronize(e1);
            if (err == cudaSuccess) err = cudaGetLastError();
            const double per_thread = (double)YS_ITERS * YS_CHAINS;
            work = which == 0 ? 2.0 * per_thread * grid * 256.0 * reps                 // one FMA = 2 flop per thread
                              : 512.0 * per_thread * grid * 8.0 * reps;                // one DMMA.8x8x4 = 512 flop per warp
        }
    }
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (err != cudaSuccess) { risp_set_error(ctx, std::string("risp_debug_yardstick: ") + cudaGetErrorString(err)); return err == cudaErrorMemoryAllocation ? RISP_ENOMEM : RISP_ECUDA; }
    *out = work / ((double)ms * 1e-3);
    return RISP_OK;
}
