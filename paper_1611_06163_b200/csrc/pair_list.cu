// pair_list.cu — SURVEY §8(f) row 1: the neighbour list reused over several steps (PAPER.md:136-138 construction and
// transposed layout, "Neighbor lists were updated every 5 steps").
//   k_list_decide   after the drift of every step: re-bin and rebuild the list iff twice the largest displacement since
//                   the last binning exceeds the skin (then some pair inside a cutoff could be missing from the list)
//   k_build_list    at a binning: every particle scans its 27-cell stencil (cells of edge >= cutoff + skin) and writes
//                   the candidates within cutoff + skin as 16-bit entries (neighbour run << 11 | offset), the same
//                   encoding the pair kernel's hit stacks use, into its column of the tile [tile of 256 slots][entry]
//                   [lane]: no atomics, no inter-thread communication, coalesced reads by the pair kernel.
//                   Pairs that can never interact are left out: the particle itself, and vertices of its own
//                   membrane (R16).
// The list is consumed by k_pair<..., LIST = true> (pair_kernel.cuh), which re-tests every entry against the true
// cutoffs with this step's positions.
#include "pair_kernel.cuh"

namespace {

__global__ void k_list_decide(uint32_t* __restrict__ ctl, float skin2) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const float d2 = __uint_as_float(ctl[TD_CTL_DMAX2]);
  // a pair inside a cutoff now was within cutoff + |d_i| + |d_j| at the binning: safe while 2 d_max <= skin
  const bool rebuild = ctl[TD_CTL_FORCE] != 0u || !(4.0f * d2 <= skin2);
  ctl[TD_CTL_REBUILD] = rebuild ? 1u : 0u;
  ctl[TD_CTL_FORCE] = 0u;
  ctl[TD_CTL_DMAX2] = 0u;
  ctl[TD_CTL_NDECIDE] += 1u;
  if (rebuild) ctl[TD_CTL_NREBUILD] += 1u;
}

__global__ void __launch_bounds__(256) k_build_list(const __grid_constant__ DevParams P, const PairArgs A,
                                                    const uint32_t* __restrict__ gate) {
  if (gate && gate[TD_CTL_REBUILD] == 0u) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NT = blockDim.x, t = threadIdx.x;
  const PairSmem sm = td_pair_carve(smem_raw);
  const int64_t n = A.n;
  const int64_t i0 = (int64_t)blockIdx.x * NT, i = i0 + t;
  const bool active = i < n;
  const int64_t ilast = (i0 + NT < n ? i0 + NT : n) - 1;
  const uint32_t r_first = __ldg(&A.keys[i0]), r_last = __ldg(&A.keys[ilast]);
  const uint32_t ri = active ? __ldg(&A.keys[i]) : 0xFFFFFFFFu;
  const int64_t is = active ? i : i0;
  const float4 p = __ldg(&A.rec.P4[is]);
  const uint32_t mk = __float_as_uint(__ldg(&A.rec.R8[2 * is + 1].w));
  const bool memb = P.excl_same && mk != 0u;  // a membrane vertex: candidates of the same membrane are left out
  const float rl2 = A.rlist2;
  const uint32_t cap = (uint32_t)A.nl_cap;
  uint16_t* const col = A.nlist + ((size_t)(i0 >> 8) * cap) * 256 + (size_t)t;

  for (uint32_t rb = r_first; rb <= r_last; rb += MAXLOC) {
    const int nloc = (int)min((uint32_t)MAXLOC, r_last - rb + 1u);
    __syncthreads();
    td_pair_fill_table(P, A, sm, rb, nloc, t, NT);
    __syncthreads();
    if (!(active && ri >= rb && ri - rb < (uint32_t)nloc)) continue;
    const int lc27 = (int)(ri - rb) * 27;
    const int myn = sm.tn[lc27 / 27];
    uint32_t cnt = 0;
    for (int c = 0; c < myn; ++c) {
      const float4 te = sm.tso[lc27 + c];
      const uint32_t first = __float_as_uint(te.x), ecnt = sm.tcnt[lc27 + c];
      const float4* __restrict__ src = A.rec.P4 + first;
      const float xs = p.x - te.y, ys = p.y - te.z, zs = p.z - te.w;
      const uint32_t eself = (uint32_t)i - first;  // offset of the particle itself inside this run (if it is in it)
      const uint32_t tag = (uint32_t)c << OFFBITS;
#pragma unroll 8
      for (uint32_t e = 0; e < ecnt; ++e) {
        const float4 pj = __ldg(&src[e]);
        const float dx = xs - pj.x, dy = ys - pj.y, dz = zs - pj.z;
        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        bool hit = r2 < rl2 && e != eself;
        if (hit && memb) hit = __float_as_uint(__ldg(&A.rec.R8[2 * (size_t)(first + e) + 1].w)) != mk;
        if (hit) {
          if (cnt < cap) col[(size_t)cnt * 256] = (uint16_t)(tag | e);
          ++cnt;
        }
      }
    }
    if (cnt > cap) { cnt = cap; atomicOr(A.err, TD_ERR_LIST_OVERFLOW); }
    A.nl_cnt[i] = cnt;
  }
}
}  // namespace

void td_launch_list_decide(uint32_t* ctl, float skin2, cudaStream_t st) { k_list_decide<<<1, 32, 0, st>>>(ctl, skin2); }

int td_launch_build_list(const DevParams& P, const PairArgs& A, const uint32_t* gate, cudaStream_t st) {
  if (A.n == 0) return 0;
  const size_t smem = td_pair_table_bytes();
  cudaError_t e = cudaFuncSetAttribute(k_build_list, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  k_build_list<<<(int)((A.n + 255) / 256), 256, smem, st>>>(P, A, gate);
  return 0;
}
