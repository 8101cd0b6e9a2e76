// tu_hybrid.cu -- instantiations and launchers of k_nll_hybrid (hybrid.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "hybrid.cuh"

int mipwa_hybrid_tiles_per_block(int rc) { return MIPWA_HYB_PTS(rc) * MIPWA_HYB_BLOCK / MIPWA_TILE; }

bool mipwa_hybrid_supported(int f1, int f2, int rc)
{
    bool supported = true;
    MIPWA_DISPATCH_HYB(f1, f2, rc, ((void)R1, (void)R2, (void)RCT));
    return supported;
}

cudaError_t mipwa_occupancy_nll_hybrid(int f1, int f2, int rc, int fl, int* blocks_per_sm)
{
    bool supported = true;
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_HYBFL(f1, f2, rc, fl,
                         e = cudaFuncSetAttribute(k_nll_hybrid<R1, R2, RCT, FL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                  (int)mipwa_hyb_ring_bytes(RCT));
                         if (e == cudaSuccess)
                             e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, k_nll_hybrid<R1, R2, RCT, FL>,
                                                                               MIPWA_HYB_BLOCK, mipwa_hyb_ring_bytes(RCT)));
    return supported ? e : cudaErrorInvalidValue;
}

cudaError_t mipwa_launch_nll_hybrid(int f1, int f2, int rc, int fl, int grid, cudaStream_t st, const DevModel& m,
                                    const HybCoef& cc, const double2* ev_cache, const unsigned short* eseg,
                                    long long n_ev, const double2* nm_cache, const double* gw,
                                    const unsigned short* gseg, long long n_norm, double2* partials,
                                    unsigned int* ticket, double* result, long long tag, bool overlapped)
{
    bool supported = true;
    // overlapped (mipwa_nll_batch, vectors 1..): programmatic stream serialisation, as for k_nll_recompute (kernels.cuh)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(MIPWA_HYB_BLOCK); cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = overlapped ? 1 : 0;
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_HYBFL(f1, f2, rc, fl,
                         (cfg.dynamicSmemBytes = mipwa_hyb_ring_bytes(RCT),
                          e = cudaLaunchKernelEx(&cfg, k_nll_hybrid<R1, R2, RCT, FL>, m, cc, ev_cache, eseg, n_ev, nm_cache, gw,
                                                 gseg, n_norm, partials, ticket, result, tag)));
    if (!supported) return cudaErrorInvalidValue;
    return e != cudaSuccess ? e : cudaGetLastError();
}
