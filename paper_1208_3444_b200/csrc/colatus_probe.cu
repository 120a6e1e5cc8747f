// colatus_probe.cu -- libcolatus_probe (include/colatus_probe.h): device microbenchmarks behind DESIGN.md 6.1-6.2.
// Separate from libcolatus.so on purpose: the product ABI carries no benchmark code.
#include <cuda_runtime.h>

#include "../../include/colatus_probe.h"
#include "probe_kernels.cuh"

namespace {

using namespace colatus;

struct Probe {
    float *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int sm_count = 0, clock_khz = 0;
    bool ok = false;
    explicit Probe(int device) {
        if (cudaSetDevice(device) != cudaSuccess) return;
        if (cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return;
        if (cudaDeviceGetAttribute(&clock_khz, cudaDevAttrClockRate, device) != cudaSuccess) return;
        if (cudaMalloc(&sink, 256) != cudaSuccess) return;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return;
        ok = true;
    }
    ~Probe() {
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
        if (sink) cudaFree(sink);
    }
    // best of three timed launches after one warm-up; < 0 on error
    template <typename Launch>
    float best_ms(Launch launch) {
        float best = 0.f;
        for (int r = 0; r < 4; ++r) {
            cudaEventRecord(e0, nullptr);
            launch();
            cudaEventRecord(e1, nullptr);
            if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) return -1.f;
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) return -1.f;
            if (r > 0 && (best == 0.f || ms < best)) best = ms;
        }
        return best;
    }
};

}  // namespace

extern "C" int colatus_probe_fp32_peak(int device, int packed, double *tflops, double *ms_out) {
    if (!tflops) return -1;
    Probe p(device);
    if (!p.ok) return -2;
    const int blocks = p.sm_count * 8 * 16;                    // 16 full waves of 8 CTAs/SM
    float *sink = p.sink;
    const float ms = p.best_ms([&] {
        if (packed)
            calibrate_fma_kernel<1><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink);
        else
            calibrate_fma_kernel<0><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink);
    });
    if (ms <= 0.f) return -2;
    const double lane_fma = (double)blocks * CAL_THREADS * (double)CAL_ITERS * CAL_CHAINS * 2.0;   // per launch
    *tflops = 2.0 * lane_fma / ((double)ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    return 0;
}

extern "C" int colatus_probe_pipe(int device, int mode, double *cycles_per_group) {
    if (!cycles_per_group || mode < 0 || mode > 7) return -1;
    Probe p(device);
    if (!p.ok) return -2;
    const int blocks = p.sm_count * 8 * 8;                      // 8 full waves of 8 CTAs/SM (16 warps per SMSP)
    float *sink = p.sink;
    const float ms = p.best_ms([&] {
        switch (mode) {
            case 0: pipe_probe_kernel<0><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            case 1: pipe_probe_kernel<1><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            case 2: pipe_probe_kernel<2><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            case 3: pipe_probe_kernel<3><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            case 4: pipe_probe_kernel<4><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            case 5: pipe_probe_kernel<5><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            case 6: pipe_probe_kernel<6><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
            default: pipe_probe_kernel<7><<<blocks, CAL_THREADS>>>(0.999f, 0.001f, sink); break;
        }
    });
    if (ms <= 0.f) return -2;
    const double groups_per_smsp = (double)blocks * (CAL_THREADS / 32) * PROBE_GROUPS / ((double)p.sm_count * 4.0);
    *cycles_per_group = (double)ms * 1e-3 * (double)p.clock_khz * 1e3 / groups_per_smsp;   // at the max SM clock
    return 0;
}
