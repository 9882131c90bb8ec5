// pair_l1.cu — the pair kernel fed from the reused neighbour list, 1 thread per particle (see pair_kernel.cuh)
#include "pair_kernel.cuh"

int td_launch_pair_l1(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  return launch_split<1, true>(P, A, nthreads, st);
}
