// librpa_probes.so -- issue-rate probes of the B200 units the chi0 path is bound by (include/rpa_probes.h).
// MEASUREMENT code for bench.py only: it is not part of librpa_chi0.so, takes no handle and allocates (and frees) its own
// few bytes of device memory.  The rooflines bench.py reports for the rank-K update divide by what
// these kernels reach: register-only mma.sync.m8n8k4.f64 on every SM (FP64 tensor pipe) and tcgen05.mma.kind::i8 from one
// thread per SM (int8 tensor pipe).
#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdio.h>

#include <algorithm>
#include <vector>

#include "../../include/rpa_probes.h"
#include "probe_i8.cuh"

namespace {
thread_local char g_perr[512] = "";
int pfail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_perr, sizeof(g_perr), fmt, ap);
    va_end(ap);
    return code;
}
#define CUDA_TRY(expr)                                                                                      \
    do {                                                                                                    \
        cudaError_t e_ = (expr);                                                                            \
        if (e_ != cudaSuccess) return pfail(RPA_PROBE_ERR_CUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)
}  // namespace

// ---- FP64 tensor issue-rate probe -----------------------------------------------------------------------------
__global__ void dmma_probe_kernel(double *out, int iters, double a0, double b0) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) c[i][0] = c[i][1] = 0.0;
    const double a = a0 + threadIdx.x * 1e-9, b = b0;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;  // never true: keeps the loop alive without memory traffic
}

extern "C" {

const char *rpa_probe_last_error(void) { return g_perr; }

int rpa_probe_fp64_tensor_peak(void *cuda_stream, double *tflops) {
    if (!tflops) return pfail(RPA_PROBE_ERR_INVALID_ARG, "rpa_probe_fp64_tensor_peak: NULL argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    double *buf = nullptr;
    CUDA_TRY(cudaMalloc(&buf, 64));  // the probe is the one call that allocates: it has no handle / workspace
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    const int iters = 100000, threads = 512;
    dmma_probe_kernel<<<nsm, threads, 0, st>>>(buf, 2000, 1.0, 1e-3);
    double best = 0.0;
    for (int rep = 0; rep < 3; rep++) {
        CUDA_TRY(cudaEventRecord(e0, st));
        dmma_probe_kernel<<<nsm, threads, 0, st>>>(buf, iters, 1.0, 1e-3);
        CUDA_TRY(cudaEventRecord(e1, st));
        CUDA_TRY(cudaEventSynchronize(e1));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
        const double fl = (double)nsm * (threads / 32) * (double)iters * 8.0 * 512.0;
        best = std::max(best, fl / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    *tflops = best;
    return RPA_PROBE_OK;
}

int rpa_probe_int8_tensor_peak(void *cuda_stream, double *tops, int32_t *mismatches) {
    if (!tops || !mismatches) return pfail(RPA_PROBE_ERR_INVALID_ARG, "rpa_probe_int8_tensor_peak: NULL argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    std::vector<int8_t> A(I8_M * I8_K), B(I8_N * I8_K);
    uint32_t x = 12345u;   // small LCG: values in [-64, 63]
    for (auto *v : {&A, &B})
        for (auto &e : *v) { x = x * 1664525u + 1013904223u; e = (int8_t)((int)((x >> 24) & 127) - 64); }
    unsigned char *buf = nullptr;   // like the FP64 probe: no handle, no workspace, allocates and frees its own scratch
    const size_t nD = (size_t)I8_M * I8_N * sizeof(int32_t);
    CUDA_TRY(cudaMalloc(&buf, A.size() + B.size() + nD));
    int8_t *dA = (int8_t *)buf, *dB = dA + A.size();
    int32_t *dD = (int32_t *)(buf + A.size() + B.size());
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = RPA_PROBE_OK;
    double best = 0.0;
    std::vector<int32_t> D((size_t)I8_M * I8_N);
    do {
#define PROBE_TRY(expr) if ((expr) != cudaSuccess) { rc = pfail(RPA_PROBE_ERR_CUDA, "rpa_probe_int8_tensor_peak: %s", cudaGetErrorString(cudaGetLastError())); break; }
        PROBE_TRY(cudaMemcpyAsync(dA, A.data(), A.size(), cudaMemcpyHostToDevice, st));
        PROBE_TRY(cudaMemcpyAsync(dB, B.data(), B.size(), cudaMemcpyHostToDevice, st));
        PROBE_TRY(cudaMemsetAsync(dD, 0xff, nD, st));
        PROBE_TRY(cudaEventCreate(&e0));
        PROBE_TRY(cudaEventCreate(&e1));
        i8_probe_kernel<<<nsm, 128, 0, st>>>(dA, dB, dD, 100);
        PROBE_TRY(cudaMemcpyAsync(D.data(), dD, nD, cudaMemcpyDeviceToHost, st));
        const int iters = 20000;
        for (int rep = 0; rep < 3 && rc == RPA_PROBE_OK; rep++) {
            PROBE_TRY(cudaEventRecord(e0, st));
            i8_probe_kernel<<<nsm, 128, 0, st>>>(dA, dB, dD, iters);
            PROBE_TRY(cudaEventRecord(e1, st));
            PROBE_TRY(cudaEventSynchronize(e1));
            float ms = 0.f;
            PROBE_TRY(cudaEventElapsedTime(&ms, e0, e1));
            best = std::max(best, (double)nsm * (iters + 1.0) * 2.0 * I8_M * I8_N * I8_K / (ms * 1e-3) * 1e-12);
        }
#undef PROBE_TRY
    } while (0);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (rc != RPA_PROBE_OK) return rc;
    int bad = 0;
    for (int i = 0; i < I8_M; i++)
        for (int j = 0; j < I8_N; j++) {
            int32_t sum = 0;
            for (int k = 0; k < I8_K; k++) sum += (int32_t)A[i * I8_K + k] * (int32_t)B[j * I8_K + k];
            bad += sum != D[(size_t)i * I8_N + j];
        }
    *mismatches = bad;
    *tops = best;
    return RPA_PROBE_OK;
}

}  // extern "C"
