// microbench.cu -- cgtp_fma_peak: the measured FP32 FMA-pipe rate that the "alu" roofline of the on-site path is
// reported against.  Register-only dependent chains: no memory traffic, no shared memory, so the
// rate is what the FFMA / FFMA2 issue path sustains at the clock the box runs under this load.
#include "common.cuh"

namespace cgtp {

constexpr int kChains = 16;   // independent accumulators per thread (latency 4 x issue rate 1/2 needs >= 2 per warp; 16 leaves slack)
constexpr int kInner = 64;    // FMAs per chain and outer iteration

template <bool PACKED>
__global__ void __launch_bounds__(256) fma_peak_kernel(float* sink, int outer, float a, float b)
{
    float2 acc[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) acc[k] = make_float2(threadIdx.x * 1e-6f + k, k * 0.5f);
    const float2 a2 = make_float2(a, a * 0.999f), b2 = make_float2(b, b * 1.001f);
    for (int it = 0; it < outer; ++it) {
#pragma unroll
        for (int j = 0; j < kInner; ++j) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) {
                if (PACKED) {
                    acc[k] = __ffma2_rn(acc[k], a2, b2);
                } else {
                    acc[k].x = fmaf(acc[k].x, a, b);
                    acc[k].y = fmaf(acc[k].y, a2.y, b2.y);
                }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += acc[k].x + acc[k].y;
    if (s == 12345.678f) sink[0] = s;  // keeps the chains alive; never true for these operands in practice
}

}  // namespace cgtp

using namespace cgtp;

extern "C" int cgtp_fma_peak(int packed, double ms_target, double* tflops, double* sm_mhz_est, void* cuda_stream)
{
    clear_error();
    if (!tflops || (packed != 0 && packed != 1) || !(ms_target > 0.0) || ms_target > 2000.0) {
        set_error("cgtp_fma_peak: invalid argument");
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    float* sink = nullptr;
    CGTP_CUDA_CHECK(cudaMalloc(&sink, 16));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = CGTP_OK;
    auto cleanup = [&]() {
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
        cudaFree(sink);
    };
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        set_error("cgtp_fma_peak: event creation failed");
        cleanup();
        return CGTP_ERR_CUDA;
    }
    const int sms = num_sms();
    const int grid = sms * 4, block = 256;
    auto run = [&](int outer, float* ms) -> cudaError_t {
        cudaEventRecord(e0, st);
        {
            LaunchScope scope(K_MISC, st);
            if (packed) fma_peak_kernel<true><<<grid, block, 0, st>>>(sink, outer, 0.9999f, 1e-4f);
            else fma_peak_kernel<false><<<grid, block, 0, st>>>(sink, outer, 0.9999f, 1e-4f);
        }
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
        return e;
    };
    // flop of one launch: every thread runs outer * kInner * kChains FMAs on 2 lanes (packed or as two scalar FMAs)
    auto flop = [&](int outer) { return 2.0 * 2.0 * (double)kChains * kInner * outer * (double)grid * block; };
    float ms = 0.f;
    cudaError_t e = run(64, &ms);  // warm-up and calibration
    if (e == cudaSuccess) e = run(64, &ms);
    if (e == cudaSuccess) {
        int outer = (int)(64.0 * ms_target / (ms > 1e-3f ? ms : 1e-3f));
        if (outer < 64) outer = 64;
        if (outer > (1 << 22)) outer = 1 << 22;
        e = run(outer, &ms);
        if (e == cudaSuccess) {
            *tflops = flop(outer) / (ms * 1e-3) * 1e-12;
            if (sm_mhz_est) *sm_mhz_est = *tflops * 1e12 / ((double)sms * 128.0 * 2.0) * 1e-6;
        }
    }
    if (e != cudaSuccess) {
        set_error("cgtp_fma_peak: %s", cudaGetErrorString(e));
        rc = CGTP_ERR_CUDA;
    }
    cleanup();
    return rc;
}
