// vn_peaks.cu -- measured issue rates of the pipes that bound the pair kernels (vn_pipe_peaks).
//
// The far-field path is bound by the plain ALU pipes, for which MEASURED_PEAKS.json has no entry (it holds the
// HBM copy bandwidth and the bf16 tensor throughput).  SURVEY.md section 8d asks for the nominal lane counts to
// be "confirmed by microbenchmark"; this file is that microbenchmark, shipped in the library so that bench.py
// measures the roofline denominator in the same run, on the same clocks, as the kernels it judges:
//   FFMA2  fma.rn.f32x2 streams (the packed fp32 instruction of sm_100 the fp32 pair kernel is made of)
//   FFMA   fma.rn.f32 streams
//   MUFU   rcp.approx + lg2.approx streams (the two SFU operations of the pair kernel)
//   DFMA   fma.rn.f64 streams (the fp64 pair kernel)
// Each kernel runs kChains independent dependency chains per thread (register operands only, no memory traffic
// inside the loop) with enough warps per SM to cover the pipe latency; several launch shapes are tried and the
// best rate is returned, in lane-operations per second (an FFMA2 thread-instruction counts as two).
#include "vn_common.cuh"

namespace vn {

constexpr int kChains = 8;
constexpr int kInner = 16;      // chain steps per loop iteration (unrolled)

__global__ void __launch_bounds__(256) peak_ffma2_kernel(int iters, float b, float c, float *sink)
{
    u64 a[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) a[k] = pk(1.0f + 0.001f * (float)(threadIdx.x + k), 0.5f + 0.002f * (float)k);
    const u64 bb = pk(b, b), cc = pk(c, c);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kInner; ++u) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fma2(a[k], bb, cc);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        float lo, hi;
        upk(a[k], lo, hi);
        s += lo + hi;
    }
    if (s == 123.456f) sink[0] = s;             // never true for the constants used; keeps the chains alive
}

__global__ void __launch_bounds__(256) peak_ffma_kernel(int iters, float b, float c, float *sink)
{
    float a[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) a[k] = 1.0f + 0.001f * (float)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kInner; ++u) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fmaf(a[k], b, c);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += a[k];
    if (s == 123.456f) sink[0] = s;
}

// rcp chains are self-stable (x -> 1/x -> x); lg2 chains are mapped back into [3, 4] by one FFMA each (the FMA
// pipe has eight times the SFU's lanes, so it is never what this kernel waits for)
__global__ void __launch_bounds__(256) peak_mufu_kernel(int iters, float one, float two, float *sink)
{
    float x[kChains / 2], y[kChains / 2];
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) {
        x[k] = 1.5f + 0.001f * (float)(threadIdx.x + k);
        y[k] = 3.0f + 0.001f * (float)(threadIdx.x & 31) + 0.1f * (float)k;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kInner; ++u) {
#pragma unroll
            for (int k = 0; k < kChains / 2; ++k) {
                x[k] = sfu_rcp(x[k]);
                y[k] = fmaf(sfu_lg2(y[k]), one, two);     // lg2 of [3,4] lies in [1.58, 2]; + 2 -> [3.58, 4]
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) s += x[k] + y[k];
    if (s == 123.456f) sink[0] = s;
}

__global__ void __launch_bounds__(256) peak_dfma_kernel(int iters, double b, double c, float *sink)
{
    double a[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) a[k] = 1.0 + 0.001 * (double)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kInner; ++u) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fma(a[k], b, c);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += a[k];
    if (s == 123.456) sink[0] = (float)s;
}

// The streams above re-read two of their three operands from one instruction to the next (register-reuse cache
// hits).  These two read three DIFFERENT register pairs in every instruction and share no operand slot with their
// neighbours -- the operand pattern of a kernel whose inputs change every instruction -- and measure what the
// register file can feed the pipes in that case.
__global__ void __launch_bounds__(256) peak_ffma2_noreuse_kernel(int iters, float b0, float c0, float *sink)
{
    u64 a[kChains], b[kChains], c[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        a[k] = pk(1.0f + 0.001f * (float)(threadIdx.x + k), 0.5f + 0.002f * (float)k);
        b[k] = pk(b0 - 0.0001f * (float)k, b0 - 0.0002f * (float)k);
        c[k] = pk(c0 + 0.0001f * (float)k, c0 + 0.0002f * (float)k);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kInner; ++u) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fma2(a[k], b[(k + u) % kChains], c[(k + 3 * u + 1) % kChains]);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        float lo, hi;
        upk(a[k], lo, hi);
        s += lo + hi;
    }
    if (s == 123.456f) sink[0] = s;
}

__global__ void __launch_bounds__(256) peak_dfma_noreuse_kernel(int iters, double b0, double c0, float *sink)
{
    double a[kChains], b[kChains], c[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        a[k] = 1.0 + 0.001 * (double)(threadIdx.x + k);
        b[k] = b0 - 0.0001 * (double)k;
        c[k] = c0 + 0.0001 * (double)k;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kInner; ++u) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fma(a[k], b[(k + u) % kChains], c[(k + 3 * u + 1) % kChains]);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += a[k];
    if (s == 123.456) sink[0] = (float)s;
}

// rates[0..3] = FFMA2, FFMA, MUFU (rcp + lg2), DFMA lane-operations per second; rates[4] = SM count of the device;
// rates[5], rates[6] = FFMA2 and DFMA streams without operand reuse; rates[7] = 0 (reserved)
vn_status pipe_peaks(double *rates, cudaStream_t st)
{
    int dev = 0, sms = 0;
    VN_CUDA(cudaGetDevice(&dev));
    VN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *sink = nullptr;
    VN_CUDA(cudaMallocAsync((void **)&sink, 16, st));
    cudaEvent_t e0, e1;
    VN_CUDA(cudaEventCreate(&e0));
    VN_CUDA(cudaEventCreate(&e1));
    vn_status rc = VN_OK;
    // launch shapes: (threads per block, blocks per SM): 16, 32 and 64 warps per SM
    const int shapes[3][2] = {{128, 4}, {256, 4}, {256, 8}};
    const int slot_of[6] = {0, 1, 2, 3, 5, 6};
    rates[7] = 0.0;
    for (int kind = 0; kind < 6 && rc == VN_OK; ++kind) {
        // about a millisecond per launch at nominal rates
        const int iters = (kind == 0 || kind == 1 || kind == 4) ? 2048 : (kind == 2 ? 512 : 1024);
        const double lane_ops_per_thread = (double)iters * kInner * kChains * ((kind == 0 || kind == 4) ? 2.0 : 1.0);
        double best = 0.0;
        for (int sh = 0; sh < 3 && rc == VN_OK; ++sh) {
            const int threads = shapes[sh][0], blocks = shapes[sh][1] * sms;
            for (int rep = 0; rep < 3; ++rep) {          // the first repetition warms up
                if (rep > 0) cudaEventRecord(e0, st);
                switch (kind) {
                    case 0: peak_ffma2_kernel<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
                    case 1: peak_ffma_kernel<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
                    case 2: peak_mufu_kernel<<<blocks, threads, 0, st>>>(iters, 1.0f, 2.0f, sink); break;
                    case 3: peak_dfma_kernel<<<blocks, threads, 0, st>>>(iters, 0.999, 0.001, sink); break;
                    case 4: peak_ffma2_noreuse_kernel<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
                    default: peak_dfma_noreuse_kernel<<<blocks, threads, 0, st>>>(iters, 0.999, 0.001, sink); break;
                }
                count_launch(1);
                if (rep > 0) {
                    cudaEventRecord(e1, st);
                    float ms = 0.f;
                    if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess ||
                        !(ms > 0.f)) {
                        rc = VN_ERR_CUDA;
                        break;
                    }
                    const double rate = lane_ops_per_thread * (double)threads * (double)blocks / ((double)ms * 1e-3);
                    if (rate > best) best = rate;
                }
            }
        }
        rates[slot_of[kind]] = best;
    }
    rates[4] = (double)sms;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (cudaGetLastError() != cudaSuccess) rc = VN_ERR_CUDA;
    VN_CUDA(cudaFreeAsync(sink, st));
    VN_CUDA(cudaStreamSynchronize(st));
    return rc;
}

}  // namespace vn
