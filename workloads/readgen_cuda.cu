// readgen_cuda.cu — device twin of the synthetic read generator (see readgen_core.h). Input generation
// only: writes ASCII reads straight into HBM so large configs never cross PCIe. C ABI, plain pointers.
#include "readgen_core.h"
#include <cuda_runtime.h>

__global__ void rg_generate_kernel(rg_params p, const uint64_t *__restrict__ glen, const uint64_t *__restrict__ cdf,
                                   uint64_t r0, uint64_t n, char *__restrict__ out) {
    // one warp per read: lane 0 resolves the header, lanes stride over the bases
    const uint32_t lane = threadIdx.x & 31;
    const uint64_t warp = (uint64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const uint64_t nwarps = (uint64_t)gridDim.x * (blockDim.x >> 5);
    for (uint64_t i = warp; i < n; i += nwarps) {
        rg_read h = rg_read_header(&p, glen, cdf, r0 + i);
        char *o = out + i * (uint64_t)p.read_len;
        for (uint32_t j = lane; j < p.read_len; j += 32) o[j] = rg_read_letter(&p, &h, j);
    }
}

// All pointers are DEVICE pointers. Returns the cudaError_t as int. Asynchronous on `stream`.
extern "C" int rg_generate_device(const rg_params *p, const uint64_t *d_glen, const uint64_t *d_cdf,
                                  uint64_t r0, uint64_t r1, char *d_out, void *stream) {
    if (r1 <= r0) return 0;
    uint64_t n = r1 - r0;
    uint64_t blocks = (n + 7) / 8;
    if (blocks > 148 * 64) blocks = 148 * 64;
    rg_generate_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(*p, d_glen, d_cdf, r0, n, d_out);
    return (int)cudaGetLastError();
}
