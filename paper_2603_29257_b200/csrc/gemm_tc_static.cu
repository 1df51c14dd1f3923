// gemm_tc_static.cu -- risp_tcgemm_static: the single-precision-mode GEMM of gemm_tc.cu (Eq. 22-23 on the tcgen05 tensor cores,
// PAPER.md:163-167, 201) for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  The allocating form (risp_debug_tcgemm) takes its bf16 operand planes from cudaMalloc on every call; here
// they live in ONE file-scope device array of RISP_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit.
//
// In host code the name of a __device__ array is a host-side stand-in, not a device address: the address the kernels (and the TMA
// tensor maps) need comes from cudaGetSymbolAddress, asked once per device with that device current, below.
//
// All calls share the array and it keeps the contents of the last call.  Nothing has to start at zero beyond what a call writes
// itself: the split kernel writes every element of the planes the GEMM reads, padding columns included, and rows beyond M / N are
// zero-filled by the TMA bounds.  Calls that overlap on the GPU (two streams, or two host threads without ordering) race on it.
#include "common.cuh"
#include <cstdarg>
#include <mutex>

static __device__ __align__(256) unsigned char g_static_scratch[RISP_STATIC_SCRATCH_BYTES];

namespace {

std::mutex g_mu;
void *g_scratch_ptr[64] = {};              // device address of g_static_scratch, per device ordinal
thread_local char g_err[256] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

// once per device, with that device current
int scratch_address(int dev, void **out)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return fail(RISP_ECUDA, "risp_tcgemm_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return RISP_OK;
}

}  // namespace

extern "C" const char *risp_static_last_error(void) { return g_err; }

extern "C" int risp_tcgemm_static(int32_t M, int32_t N, int32_t K, const double *A_dev, const double *B_dev, double *C_dev, int32_t accumulate,
                                  void *cuda_stream)
{
    g_err[0] = 0;
    if (M <= 0 || N <= 0 || K <= 0 || !A_dev || !B_dev || !C_dev) return fail(RISP_EINVAL, "risp_tcgemm_static: need M, N, K >= 1 and non-NULL device pointers");
    const long long ldk = ((long long)K + 7) & ~7LL;
    const long long planeA = (long long)M * ldk, planeB = (long long)N * ldk;         // elements per bf16 plane
    const unsigned long long need = 3ull * 2ull * (unsigned long long)(planeA + planeB);
    if (need > (unsigned long long)RISP_STATIC_SCRATCH_BYTES)
        return fail(RISP_EINVAL, "risp_tcgemm_static: %d x %d x %d needs %llu bytes of operand planes (6 (M + N) ceil8(K)), the static scratch holds %llu",
                    (int)M, (int)N, (int)K, need, (unsigned long long)RISP_STATIC_SCRATCH_BYTES);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return fail(RISP_ECUDA, "risp_tcgemm_static: no current device (or ordinal >= 64)");
    cudaDeviceProp prop;
    static int major[64] = {};
    if (!major[dev]) {
        if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return fail(RISP_ECUDA, "risp_tcgemm_static: cudaGetDeviceProperties failed");
        major[dev] = prop.major;
    }
    if (major[dev] != 10) return fail(RISP_EINVAL, "risp_tcgemm_static: needs the tcgen05 tensor cores (sm_100), device %d is sm_%d", dev, major[dev] * 10);
    void *base = nullptr;
    int rc = scratch_address(dev, &base);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned short *a = (unsigned short *)base;                  // bf16 bit patterns: [3][M][ldk], then [3][N][ldk]
    unsigned short *b = a + 3 * planeA;                          // 3 planeA * 2 bytes is a multiple of 48: 16-byte aligned for the tensor map
    cudaError_t e;
    if ((e = risp_split_rows_bf3(A_dev, K, M, K, a, ldk, planeA, 0, 0, st)) != cudaSuccess ||
        (e = risp_split_rows_bf3(B_dev, K, N, K, b, ldk, planeB, 0, 0, st)) != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(RISP_ECUDA, "risp_tcgemm_static: operand split failed: %s", cudaGetErrorString(e));
    }
    TcGemmDesc d;
    d.M = M; d.N = N; d.K = K; d.nb = 1;
    d.A = a; d.lda = ldk; d.planeA = planeA; d.sA = 0;
    d.B = b; d.ldb = ldk; d.planeB = planeB; d.sB = 0;
    d.C = C_dev; d.ldc = M; d.sC = 0; d.planeC = 0; d.out_kind = 0; d.rpg = 0; d.gstride = 0; d.accumulate = accumulate ? 1 : 0;
    if ((e = risp_tcgemm(d, st)) != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(RISP_ECUDA, "risp_tcgemm_static: GEMM launch failed: %s", cudaGetErrorString(e));
    }
    return RISP_OK;
}
