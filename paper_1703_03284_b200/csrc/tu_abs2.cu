// tu_abs2.cu -- instantiations and launcher of the per-point test hook k_abs2 (kernels.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"

cudaError_t mipwa_launch_abs2(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                              const double* s12, const double* s13, const unsigned short* seg, long long n, double* out)
{
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_abs2<R1, R2, FL><<<grid, MIPWA_BLOCK, 0, st>>>(m, s12, s13, seg, n, out)));
    return cudaGetLastError();
}
