// pair_s2.cu — the pair kernel with 2 threads per particle (see pair_kernel.cuh)
#include "pair_kernel.cuh"

int td_launch_pair_s2(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  return launch_split<2, false>(P, A, nthreads, st);
}
