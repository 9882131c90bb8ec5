// pair.cu — dispatch of the pair kernel (pair_kernel.cuh) over the threads-per-particle variants, each compiled in its
// own translation unit (pair_s1.cu, pair_s2.cu, pair_s4.cu, pair_s16.cu; pair_l1.cu: candidates from the neighbour list).
#include "common.cuh"

int td_launch_pair_s1(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_s2(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_s4(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_s16(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);
int td_launch_pair_l1(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st);

size_t td_pair_smem_bytes(int lcap, int nthreads) { return td_pair_table_bytes() + (size_t)lcap * nthreads * 2; }

int td_launch_pair(const DevParams& P, const PairArgs& A, int nthreads, int split, bool from_list, cudaStream_t st) {
  if (from_list) return td_launch_pair_l1(P, A, nthreads, st);
  if (split >= 16) return td_launch_pair_s16(P, A, nthreads, st);
  if (split >= 4) return td_launch_pair_s4(P, A, nthreads, st);
  if (split >= 2) return td_launch_pair_s2(P, A, nthreads, st);
  return td_launch_pair_s1(P, A, nthreads, st);
}
