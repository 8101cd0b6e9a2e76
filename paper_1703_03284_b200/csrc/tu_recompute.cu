// tu_recompute.cu -- instantiations and launchers of k_nll_recompute (kernels.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"

cudaError_t mipwa_launch_nll_recompute(const int* n_spin, int fl, bool mix, int grid, cudaStream_t st, const DevModel& m,
                                       const PointRec* ev, double kappa, long long n_ev, const PointRec* nm,
                                       long long n_norm, double2* partials, unsigned int* ticket, double* result,
                                       long long tag)
{
    if (mix)
        return mipwa_launch_nll_recompute_mix(n_spin, fl, grid, st, m, ev, kappa, n_ev, nm, n_norm, partials, ticket,
                                              result, tag, nullptr);
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_nll_recompute<R1, R2, FL, false><<<grid, MIPWA_REC_BLOCK, 0, st>>>(
                             m, ev, 0.0, n_ev, nm, n_norm, partials, ticket, result, tag, nullptr)));
    return cudaGetLastError();
}

// the same launch with programmatic stream serialisation: this kernel may start before the previous launch on the stream has
// completed (kernels.cuh: griddepcontrol in k_nll_recompute).  Only for a launch whose predecessor on the stream is the same
// kernel on the same point records (mipwa_nll_batch).
template <class... KA, class... A>
static cudaError_t launch_serialised(void (*kernel)(KA...), int grid, cudaStream_t st, A&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(MIPWA_REC_BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KA>(args)...);
}

cudaError_t mipwa_launch_nll_recompute_overlapped(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                                                  const PointRec* ev, long long n_ev, const PointRec* nm, long long n_norm,
                                                  double2* partials, unsigned int* ticket, double* result, long long tag)
{
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (e = launch_serialised(k_nll_recompute<R1, R2, FL, false>, grid, st, m, ev, 0.0, n_ev, nm, n_norm,
                                                partials, ticket, result, tag, (const double*)nullptr)));
    return e != cudaSuccess ? e : cudaGetLastError();
}
