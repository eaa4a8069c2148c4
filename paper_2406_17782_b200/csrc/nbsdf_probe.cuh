// nbsdf_probe.cuh -- DEBUG instrumentation, compiled only with -DNBSDF_PROBE (python -m paper_2406_17782_b200.probe builds
// a separate libnbsdf_probe.so; the product library never contains any of this).  A few threads of every CTA stamp
// (SM clock, global timer) at fixed points of the kernel; stamps are keyed by (launch % 32, SM id), so the gap between
// consecutive launches on one SM, the prologue, the pipeline fill and the drain can be read back per SM.
#pragma once
#ifdef NBSDF_PROBE
#include <cuda_runtime.h>
#include <stdint.h>

namespace nbsdf {

constexpr int kProbeLaunches = 32, kProbeSms = 160, kProbeStamps = 10;
__device__ unsigned long long g_probe[kProbeLaunches][kProbeSms][kProbeStamps][2];

__device__ __forceinline__ void probe_stamp(int launch, int stamp)
{
    unsigned smid;
    unsigned long long gt;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
    unsigned long long* p = g_probe[launch & (kProbeLaunches - 1)][smid < kProbeSms ? smid : kProbeSms - 1][stamp];
    p[0] = (unsigned long long)clock64();
    p[1] = gt;
}

}  // namespace nbsdf

// out: kProbeLaunches * kProbeSms * kProbeStamps * 2 uint64; synchronises the device first
extern "C" int nbsdf_debug_read_probe(unsigned long long* out)
{
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return (int)e;
    return (int)cudaMemcpyFromSymbol(out, nbsdf::g_probe, sizeof(nbsdf::g_probe));
}
extern "C" int nbsdf_debug_clear_probe()
{
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, nbsdf::g_probe);
    if (e != cudaSuccess) return (int)e;
    return (int)cudaMemset(p, 0, sizeof(nbsdf::g_probe));
}
#define NBSDF_STAMP(cond, net, i) do { if (cond) nbsdf::probe_stamp((net).probe_slot, (i)); } while (0)
#else
#define NBSDF_STAMP(cond, net, i) do { } while (0)
#endif
