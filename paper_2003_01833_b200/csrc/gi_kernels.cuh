// gi_kernels.cuh -- launchers of the Green-Iteration epilogue (Algorithm 2 lines 4-7).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace bltc {

// layout of the result vector of bltc_gi_update (include/bltc.h)
enum { kGiEpsNew = 0, kGiDelta = 1, kGiNorm = 2, kGiResidual = 3, kGiCoeff = 4 };

// records `msg` as the calling thread's bltc_last_error() and returns `code` (defined in api.cu)
int set_last_error(int code, const char* msg);

int gi_grid_blocks(int64_t n, int sm_count);
size_t gi_scratch_doubles(int n_prev, int nblk);

// All pointers are device pointers.  psi_new is updated in place (orthogonalised, normalised).
// result: [4 + n_prev] doubles; scratch: gi_scratch_doubles(n_prev, nblk) doubles.
cudaError_t launch_gi_update(const double* w, const double* psi_old, const double* f_old, double* psi_new,
                             const double* phi, int n_prev, int64_t n, double eps_old, double* result,
                             double* scratch, int nblk, cudaStream_t st);

}  // namespace bltc
