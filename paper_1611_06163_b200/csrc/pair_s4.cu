// pair_s4.cu — the pair kernel with 4 threads per particle (see pair_kernel.cuh)
#include "pair_kernel.cuh"

int td_launch_pair_s4(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  return launch_split<4, false>(P, A, nthreads, st);
}
