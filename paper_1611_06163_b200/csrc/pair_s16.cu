// pair_s16.cu — the pair kernel with 16 threads per particle (see pair_kernel.cuh)
#include "pair_kernel.cuh"

int td_launch_pair_s16(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  return launch_split<16, false>(P, A, nthreads, st);
}
