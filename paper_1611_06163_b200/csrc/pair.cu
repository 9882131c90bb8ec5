// pair.cu — dispatch of the pair kernel (pair_kernel.cuh) over the threads-per-particle variants, each compiled in its
// own translation unit (pair_s1.cu, pair_s2.cu, pair_s4.cu, pair_s16.cu).
#include "common.cuh"

int td_launch_pair_s1(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_s2(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_s4(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_s16(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);

size_t td_pair_smem_bytes(int lcap, int nthreads) {
  return (size_t)TD_PAIR_MAXLOC * 27 * 20 + 8 * 16 * 4 + TD_PAIR_MAXLOC * 4 + (size_t)lcap * nthreads * 2;
}

int td_launch_pair(const DevParams& P, const PairArgs& A, int nthreads, int split, cudaStream_t st) {
  if (split >= 16) return td_launch_pair_s16(P, A, nthreads, st);
  if (split >= 4) return td_launch_pair_s4(P, A, nthreads, st);
  if (split >= 2) return td_launch_pair_s2(P, A, nthreads, st);
  return td_launch_pair_s1(P, A, nthreads, st);
}
