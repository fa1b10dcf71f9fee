// bege_probe.cu -- measurement probes that are NOT part of the product: built into their own library
// (libbege_probe.so, C ABI in include/bege_probe.h) so that the search library and its public header carry no experiment.
// Today: the overlap-save bake-off of SURVEY.md 8(f) NEXT #4 (csrc/ovs_probe.cuh; decision in DESIGN.md section 8).
#include <algorithm>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/bege.h"
#include "../../include/bege_probe.h"
#include "ovs_probe.cuh"

using namespace bege;

// ------------------------------------------------------------------------------------------------
// bake-off probe of the overlap-save variant (csrc/ovs_probe.cuh).  Self-contained: own device
// memory, own stream.  h16: T x 16384 complex template spectra (host; NULL: filled on the device with finite numbers,
// timing only), x16: n_blocks x 16384 complex block spectra (host; NULL likewise).  z_dbg (host, n_blocks x 16384 complex,
// may be NULL): the correlation blocks of template dbg_j.  *ms_out: mean time of one pass over all T x n_blocks items.
__global__ void k_ovs_fill(float2* p, uint64_t n, uint32_t seed)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        uint32_t h = (uint32_t)i * 2654435761u ^ seed; h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        p[i] = make_float2((float)(int)(h & 0xffff) * (1.0f / 65536.0f) - 0.5f, (float)(int)(h >> 16) * (1.0f / 65536.0f) - 0.5f);
    }
}

extern "C" int bege_ovs_probe(int device, uint64_t T, uint32_t n_blocks, uint32_t reps, float thr2, const float* h16,
                              const float* x16, float* z_dbg, uint64_t dbg_j, double* ms_out, uint64_t* hits_out)
{
    if (T == 0 || n_blocks == 0 || reps == 0 || !ms_out) return BEGE_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BEGE_ECUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess || prop.major < 10) return BEGE_ECUDA;
    c2 *dH = nullptr, *dX = nullptr, *dZ = nullptr; unsigned long long* dcnt = nullptr;
    const uint64_t nH = T * kOvsP, nX = (uint64_t)n_blocks * kOvsP;
    int rc = BEGE_OK;
    cudaStream_t st = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    auto done = [&](int code) {
        if (dH) cudaFree(dH); if (dX) cudaFree(dX); if (dZ) cudaFree(dZ); if (dcnt) cudaFree(dcnt);
        if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); if (st) cudaStreamDestroy(st);
        cudaGetLastError();
        return code;
    };
    if (cudaMalloc(&dH, nH * 8) != cudaSuccess || cudaMalloc(&dX, nX * 8) != cudaSuccess || cudaMalloc(&dZ, nX * 8) != cudaSuccess ||
        cudaMalloc(&dcnt, 256) != cudaSuccess) return done(BEGE_ENOMEM);
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
        cudaEventCreate(&e1) != cudaSuccess) return done(BEGE_ECUDA);
    if (h16) { if (cudaMemcpyAsync(dH, h16, nH * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return done(BEGE_ECUDA); }
    else k_ovs_fill<<<1024, 256, 0, st>>>((float2*)dH, nH, 1u);
    if (x16) { if (cudaMemcpyAsync(dX, x16, nX * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return done(BEGE_ECUDA); }
    else k_ovs_fill<<<64, 256, 0, st>>>((float2*)dX, nX, 2u);
    if (cudaMemsetAsync(dcnt, 0, 256, st) != cudaSuccess) return done(BEGE_ECUDA);
    if (cudaFuncSetAttribute(k_ovs_probe, cudaFuncAttributeMaxDynamicSharedMemorySize, kOvsSmem) != cudaSuccess) return done(BEGE_ECUDA);
    const unsigned ctas = (unsigned)std::min<uint64_t>(T * n_blocks, (uint64_t)prop.multiProcessorCount);
    int* d_abort = (int*)(dcnt + 16);
    // warm-up pass (also the one that writes z_dbg), then `reps` timed passes
    k_ovs_probe<<<ctas, 1024, kOvsSmem, st>>>(dH, dX, T, n_blocks, thr2, dcnt, z_dbg ? dZ : nullptr, dbg_j, d_abort);
    if (cudaMemsetAsync(dcnt, 0, 8, st) != cudaSuccess) return done(BEGE_ECUDA);
    cudaEventRecord(e0, st);
    for (uint32_t r = 0; r < reps; ++r)
        k_ovs_probe<<<ctas, 1024, kOvsSmem, st>>>(dH, dX, T, n_blocks, thr2, dcnt, nullptr, 0, d_abort);
    cudaEventRecord(e1, st);
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return done(BEGE_ECUDA);
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    *ms_out = (double)ms / reps;
    unsigned long long hc[17];
    if (cudaMemcpy(hc, dcnt, sizeof hc, cudaMemcpyDeviceToHost) != cudaSuccess) return done(BEGE_ECUDA);
    if (hits_out) *hits_out = hc[0] / reps;
    if (*(int*)&hc[16]) rc = BEGE_ECUDA;
    if (z_dbg && cudaMemcpy(z_dbg, dZ, nX * 8, cudaMemcpyDeviceToHost) != cudaSuccess) return done(BEGE_ECUDA);
    return done(rc);
}
