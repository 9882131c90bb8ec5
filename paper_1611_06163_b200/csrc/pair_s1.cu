// pair_s1.cu — the pair kernel with 1 thread per particle (see pair_kernel.cuh)
#include "pair_kernel.cuh"

int td_launch_pair_s1(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  return launch_split<1, false>(P, A, nthreads, st);
}
