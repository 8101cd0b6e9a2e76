// launch.h -- host launchers of the heavily specialised kernels (model signature x model flags), one translation unit
// per kernel family so that the library builds in parallel (build.py).  Internal to libmipwa.so; plain pointers only.
#pragma once
#include <cuda_runtime.h>
#include "dev_model.cuh"

struct HybCoef;

// n_spin = resonances of spin 0, 1, 2 (the kernel signature), fl = MIPWA_FL_* of the model.  Every launcher returns
// cudaGetLastError() of its launch; the occupancy functions return the resident blocks per SM of the matching kernel.

// tu_recompute.cu: k_nll_recompute; tu_abs2.cu: k_abs2 (kernels.cuh).  mix selects the mixture kernels
// (tu_recompute_mix.cu): sum of ln(|A|^2 + kappa w_i) over the event records.
cudaError_t mipwa_launch_nll_recompute(const int* n_spin, int fl, bool mix, int grid, cudaStream_t st, const DevModel& m,
                                       const PointRec* ev, double kappa, long long n_ev, const PointRec* nm,
                                       long long n_norm, double2* partials, unsigned int* ticket, double* result,
                                       long long tag);
// the same (no mixture) as a launch that may overlap the end of the previous launch on the stream (tu_recompute.cu)
cudaError_t mipwa_launch_nll_recompute_overlapped(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                                                  const PointRec* ev, long long n_ev, const PointRec* nm, long long n_norm,
                                                  double2* partials, unsigned int* ticket, double* result, long long tag);
cudaError_t mipwa_launch_nll_recompute_mix(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                                           const PointRec* ev, double kappa, long long n_ev, const PointRec* nm,
                                           long long n_norm, double2* partials, unsigned int* ticket, double* result,
                                           long long tag,
                                           const double* integral_src);
cudaError_t mipwa_launch_abs2(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                              const double* s12, const double* s13, const unsigned short* seg, long long n, double* out);

// tu_grad.cu / tu_grad_shp.cu / tu_grad_mix.cu: k_grad_recompute (grad.cuh).  smem = warps per block x 8 (N - 1)
// doubles; blocks [0, ev_blocks) take the events.  shp = 0, or 1 / 2: the first spin-1 / spin-2 device slot floats and
// its shape sums are wanted.  mix: f = -2 A / (|A|^2 + kappa w_i), partial [1] = sum w / D.
cudaError_t mipwa_grad_set_smem(const int* n_spin, int fl, bool mix, int shp, size_t smem);
cudaError_t mipwa_launch_grad_recompute(const int* n_spin, int fl, bool mix, int shp, int grid, int ev_blocks, size_t smem,
                                        cudaStream_t st, const DevModel& m, const PointRec* ev, double kappa,
                                        long long n_ev, const PointRec* nm, long long n_norm, double* partials,
                                        double2* f_ev, double2* f_nm);
cudaError_t mipwa_grad_set_smem_shp(const int* n_spin, int fl, int shp, size_t smem);
cudaError_t mipwa_launch_grad_recompute_shp(const int* n_spin, int fl, int shp, int grid, int ev_blocks, size_t smem,
                                            cudaStream_t st, const DevModel& m, const PointRec* ev, long long n_ev,
                                            const PointRec* nm, long long n_norm, double* partials);
cudaError_t mipwa_grad_set_smem_mix(const int* n_spin, int fl, size_t smem);
cudaError_t mipwa_launch_grad_recompute_mix(const int* n_spin, int fl, int grid, int ev_blocks, size_t smem,
                                            cudaStream_t st, const DevModel& m, const PointRec* ev, double kappa,
                                            long long n_ev, const PointRec* nm, long long n_norm, double* partials);

// tu_hybrid.cu: k_nll_hybrid (hybrid.cuh); f1, f2 = floating resonances of spin 1, 2, rc = cached (fixed) resonances
bool mipwa_hybrid_supported(int f1, int f2, int rc);
int mipwa_hybrid_tiles_per_block(int rc);                  // 256-point cache tiles one block takes per iteration
cudaError_t mipwa_occupancy_nll_hybrid(int f1, int f2, int rc, int fl, int* blocks_per_sm);
cudaError_t mipwa_launch_nll_hybrid(int f1, int f2, int rc, int fl, int grid, cudaStream_t st, const DevModel& m,
                                    const HybCoef& cc, const double2* ev_cache, const unsigned short* eseg,
                                    long long n_ev, const double2* nm_cache, const double* gw,
                                    const unsigned short* gseg, long long n_norm, double2* partials,
                                    unsigned int* ticket, double* result, long long tag, bool overlapped = false);
