// scmd_probe.cu -- libscmd_probe.so: context-free diagnostics (include/scmd_probe.h).  Kept out of libscmd.so so that
// the product ABI is the method and nothing else; bench.py (measured ALU peak beside the nominal one) and
// tests/test_gpu_parity.py::test_device_reciprocals (accuracy of the FP64 reciprocal building blocks) load it.
#include "../../include/scmd_probe.h"

#include <cstddef>

#include "sc_probe.cuh"

using namespace scmd;

extern "C" {

sc_status sc_probe_throughput(int32_t kind, void *cuda_stream, void *d_scratch, size_t scratch_bytes,
                              double *h_inst_per_s, double *h_sm_clock_mhz) {
    if (kind < 0 || kind > 8 || !d_scratch || !h_inst_per_s) return SC_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return SC_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = sms * 8, block = 256;
    if (scratch_bytes < sizeof(double) * 8 + sizeof(long long) * size_t(grid)) return SC_ERR_NOMEM;
    double *out = static_cast<double *>(d_scratch);
    long long *cyc = reinterpret_cast<long long *>(out + 8);
    const int iters = (kind == 3 || kind == 4) ? 2048 : 16384;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return SC_ERR_CUDA;
    auto run = [&](int it) {
        switch (kind) {
            case 0: probe_kernel<0><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 1: probe_kernel<1><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 2: probe_kernel<2><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 3: probe_kernel<3><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 4: probe_kernel<4><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 5: probe_kernel<5><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 6: probe_kernel<6><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            case 7: probe_kernel<7><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
            default: probe_kernel<8><<<grid, block, 0, st>>>(out, cyc, it, 1.0); break;
        }
    };
    run(iters / 8);   // warm-up
    run(iters);
    cudaEventRecord(e0, st);
    run(iters);
    cudaEventRecord(e1, st);
    sc_status rc = SC_OK;
    float ms = 0.f;
    long long cycles0 = 0;
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess ||
        cudaMemcpy(&cycles0, cyc, sizeof(long long), cudaMemcpyDeviceToHost) != cudaSuccess)
        rc = SC_ERR_CUDA;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc != SC_OK) return rc;
    const double per_thread = double(iters) * kProbeChains * ((kind == 2 || kind == 7 || kind == 8) ? 2.0 : 1.0);
    *h_inst_per_s = per_thread * double(grid) * block / (double(ms) * 1e-3);
    // a block's own span in SM cycles; 8 blocks per SM run concurrently, so span ~ kernel time
    if (h_sm_clock_mhz) *h_sm_clock_mhz = double(cycles0) / (double(ms) * 1e3);
    return SC_OK;
}

sc_status sc_probe_reciprocal(double lo, double hi, int32_t n_samples, void *cuda_stream, void *d_scratch,
                              size_t scratch_bytes, double *h_err4) {
    if (!(lo > 0.0) || !(hi > lo) || n_samples < 1 || !d_scratch || scratch_bytes < 4 * sizeof(double) || !h_err4)
        return SC_ERR_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double *out = static_cast<double *>(d_scratch);
    if (cudaMemsetAsync(out, 0, 4 * sizeof(double), st) != cudaSuccess) return SC_ERR_CUDA;
    reciprocal_error_kernel<<<296, 256, 0, st>>>(lo, hi, n_samples, out);
    if (cudaGetLastError() != cudaSuccess) return SC_ERR_CUDA;
    if (cudaMemcpyAsync(h_err4, out, 4 * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess) return SC_ERR_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return SC_ERR_CUDA;
    return SC_OK;
}


}  // extern "C"
