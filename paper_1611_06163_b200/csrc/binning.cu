// binning.cu — rows a2 and a3 of SURVEY §8(a): stable LSD radix sort of (cell key, previous slot) and the
// reorder + cell-start table (PAPER.md:137 "particle reordering", :141 "radix sort").  No atomics decide an
// order anywhere, so the sorted order (and with it every fp32 summation order downstream) is deterministic.
#include "common.cuh"

namespace {
constexpr int RB = 8;            // bits per pass
constexpr int NBIN = 1 << RB;
constexpr int SORT_NT = 256;     // 8 warps
constexpr int SORT_ITEMS = 16;   // keys per thread
constexpr int TILE = SORT_NT * SORT_ITEMS;
constexpr int WCHUNK = 32 * SORT_ITEMS;  // contiguous keys owned by one warp
#ifndef SORT_SCATTER_MINB
#define SORT_SCATTER_MINB 4  // 64 registers: four CTAs per SM instead of three (round 2, 6.9 M keys, three passes: 0.273 -> 0.239 ms)
#endif

// per-tile digit histogram -> hist[bin * nblk + blk]  (integer counts: atomics cannot change the result)
// `gate` (may be NULL): the device control block of the neighbour-list mode; the kernels of the binning return at once
// when this step does not re-bin (TD_CTL_REBUILD == 0), so that the launch sequence of a step stays static (CUDA graph)
#define TD_GATE(gate) if ((gate) && (gate)[TD_CTL_REBUILD] == 0u) return

__global__ void __launch_bounds__(SORT_NT) k_sort_hist(const uint32_t* __restrict__ keys, int64_t n, int shift,
                                                       uint32_t* __restrict__ hist, int nblk,
                                                       const uint32_t* __restrict__ gate) {
  TD_GATE(gate);
  __shared__ uint32_t cnt[NBIN];
  cnt[threadIdx.x] = 0;
  __syncthreads();
  // every thread takes SORT_ITEMS CONSECUTIVE keys and adds once per run of equal digits: the keys arrive almost
  // sorted (particles move little in a step), so a thread's 16 keys hold one or two digits in the low passes and the
  // 32 lanes of a warp no longer queue on one shared-memory word (config 5, three passes: sort 0.218 -> 0.196 ms; config 2: 0.056 -> 0.048 ms)
  const int64_t i0 = (int64_t)blockIdx.x * TILE + (int64_t)threadIdx.x * SORT_ITEMS;
  uint32_t k[SORT_ITEMS];
  if (i0 + SORT_ITEMS <= n && (reinterpret_cast<uintptr_t>(keys) & 15u) == 0) {  // (a caller's array may be 4-byte aligned)
#pragma unroll
    for (int q = 0; q < SORT_ITEMS / 4; ++q) {
      const uint4 v = __ldg(reinterpret_cast<const uint4*>(keys + i0) + q);
      k[4 * q] = v.x; k[4 * q + 1] = v.y; k[4 * q + 2] = v.z; k[4 * q + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int q = 0; q < SORT_ITEMS; ++q) k[q] = i0 + q < n ? keys[i0 + q] : 0u;
  }
  const int nv = (int)(n - i0 < (int64_t)SORT_ITEMS ? (n - i0 > 0 ? n - i0 : 0) : (int64_t)SORT_ITEMS);
  uint32_t dprev = 0, run = 0;
#pragma unroll
  for (int q = 0; q < SORT_ITEMS; ++q) {
    const uint32_t d = (k[q] >> shift) & (NBIN - 1);
    if (q < nv) {
      if (run && d != dprev) { atomicAdd(&cnt[dprev], run); run = 0; }
      dprev = d; ++run;
    }
  }
  if (run) atomicAdd(&cnt[dprev], run);
  __syncthreads();
  hist[(int64_t)threadIdx.x * nblk + blockIdx.x] = cnt[threadIdx.x];
}

// exclusive scan of hist[0..total) in two levels: every CTA scans one chunk of 4096 entries in place and writes the
// chunk total; k_sort_scan_tops then scans the chunk totals (one CTA); the scatter adds tops[index >> 12]
constexpr int SCAN_CHUNK = 4096;
__device__ __forceinline__ uint32_t block_excl_scan_1024(uint32_t tsum, uint32_t* wsum, uint32_t& total) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t x = tsum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t y = __shfl_up_sync(0xffffffffu, x, d);
    if (lane >= d) x += y;
  }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  if (w == 0) {
    uint32_t s = wsum[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, s, d);
      if (lane >= d) s += y;
    }
    wsum[lane] = s;  // inclusive over warps
  }
  __syncthreads();
  total = wsum[31];
  return (w ? wsum[w - 1] : 0u) + (x - tsum);
}

__global__ void __launch_bounds__(1024) k_sort_scan(uint32_t* __restrict__ hist, int64_t total,
                                                    uint32_t* __restrict__ tops, const uint32_t* __restrict__ gate) {
  TD_GATE(gate);
  __shared__ uint32_t wsum[32];
  int64_t i0 = (int64_t)blockIdx.x * SCAN_CHUNK + (int64_t)threadIdx.x * 4;
  uint32_t v[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) v[k] = (i0 + k < total) ? hist[i0 + k] : 0u;
  uint32_t sum;
  uint32_t excl = block_excl_scan_1024(v[0] + v[1] + v[2] + v[3], wsum, sum);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (i0 + k < total) hist[i0 + k] = excl;
    excl += v[k];
  }
  if (threadIdx.x == 0) tops[blockIdx.x] = gridDim.x == 1 ? 0u : sum;  // a single chunk needs no second level
}

__global__ void __launch_bounds__(1024) k_sort_scan_tops(uint32_t* __restrict__ tops, int nchunk,
                                                         const uint32_t* __restrict__ gate) {
  TD_GATE(gate);
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < nchunk; base += 1024) {
    int i = base + threadIdx.x;
    uint32_t v = i < nchunk ? tops[i] : 0u, sum;
    uint32_t excl = block_excl_scan_1024(v, wsum, sum);
    uint32_t carry = carry_s;
    if (i < nchunk) tops[i] = carry + excl;
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + sum;
    __syncthreads();
  }
}

// stable scatter: tile order = (warp, item, lane); rank = scanned tile base + keys of the same digit in earlier
// warps of the tile + earlier keys of the same digit in this warp.  The tile is first put in digit order in shared
// memory (local rank = start of the digit inside the tile + the same two terms), then written out by consecutive
// threads: keys of one digit leave as one contiguous run (~16 keys = 64 B for a uniform digit) instead of 4-byte stores
// from 32 lanes to 32 different sectors (round 2, 6.9 M keys: the three passes of a binning 0.287 -> 0.273 ms; what
// remains is the 16 MATCH.ANY per thread: replacing the shared atomics of the counting by more of them made it slower).
__global__ void __launch_bounds__(SORT_NT, SORT_SCATTER_MINB) k_sort_scatter(const uint32_t* __restrict__ kin,
                                                          const uint32_t* __restrict__ vin,
                                                          uint32_t* __restrict__ kout, uint32_t* __restrict__ vout,
                                                          int64_t n, int shift, const uint32_t* __restrict__ hist,
                                                          int nblk, const uint32_t* __restrict__ tops,
                                                          const uint32_t* __restrict__ gate) {
  TD_GATE(gate);
  __shared__ uint32_t wbase[SORT_NT / 32][NBIN];
  __shared__ uint32_t gdelta[NBIN];  // global position of a key = its position in the digit-ordered tile + gdelta[digit]
  __shared__ uint32_t wsum[SORT_NT / 32];
  __shared__ uint32_t skey[TILE], sval[TILE];
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int k = threadIdx.x; k < (SORT_NT / 32) * NBIN; k += SORT_NT) (&wbase[0][0])[k] = 0;
  __syncthreads();
  const int64_t tile0 = (int64_t)blockIdx.x * TILE;
  int64_t base = tile0 + (int64_t)w * WCHUNK;
  uint32_t key[SORT_ITEMS];
  {  // counts of this warp's 512 keys: every lane takes 16 consecutive ones and adds once per run of equal digits (as
     // in k_sort_hist); the keys are read again below in the (item, lane) order the ranks need, from L1
    const int64_t j0 = base + (int64_t)lane * SORT_ITEMS;
    if (j0 + SORT_ITEMS <= n && (reinterpret_cast<uintptr_t>(kin) & 15u) == 0) {
#pragma unroll
      for (int q = 0; q < SORT_ITEMS / 4; ++q) {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(kin + j0) + q);
        key[4 * q] = v.x; key[4 * q + 1] = v.y; key[4 * q + 2] = v.z; key[4 * q + 3] = v.w;
      }
    } else {
#pragma unroll
      for (int q = 0; q < SORT_ITEMS; ++q) key[q] = j0 + q < n ? kin[j0 + q] : 0u;
    }
    const int nv = (int)(n - j0 < (int64_t)SORT_ITEMS ? (n - j0 > 0 ? n - j0 : 0) : (int64_t)SORT_ITEMS);
    uint32_t dprev = 0, run = 0;
#pragma unroll
    for (int q = 0; q < SORT_ITEMS; ++q) {
      const uint32_t d = (key[q] >> shift) & (NBIN - 1);
      if (q < nv) {
        if (run && d != dprev) { atomicAdd(&wbase[w][dprev], run); run = 0; }
        dprev = d; ++run;
      }
    }
    if (run) atomicAdd(&wbase[w][dprev], run);
  }
#pragma unroll
  for (int it = 0; it < SORT_ITEMS; ++it) {
    int64_t i = base + it * 32 + lane;
    key[it] = i < n ? kin[i] : 0xFFFFFFFFu;
  }
  __syncthreads();
  {  // per bin (thread b owns bin b): tile count -> exclusive scan over the bins = local start of the digit
    const int b = threadIdx.x;
    uint32_t c[SORT_NT / 32], tot = 0;
#pragma unroll
    for (int ww = 0; ww < SORT_NT / 32; ++ww) { c[ww] = wbase[ww][b]; tot += c[ww]; }
    uint32_t x = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    uint32_t before = 0;
#pragma unroll
    for (int ww = 0; ww < SORT_NT / 32; ++ww) before += ww < w ? wsum[ww] : 0u;
    uint32_t run = before + x - tot;  // keys of smaller digits in this tile
    const int64_t hi = (int64_t)b * nblk + blockIdx.x;
    gdelta[b] = hist[hi] + tops[hi / SCAN_CHUNK] - run;
#pragma unroll
    for (int ww = 0; ww < SORT_NT / 32; ++ww) {
      wbase[ww][b] = run;
      run += c[ww];
    }
  }
  __syncthreads();
#pragma unroll
  for (int it = 0; it < SORT_ITEMS; ++it) {
    int64_t i = base + it * 32 + lane;
    bool valid = i < n;
    uint32_t d = valid ? ((key[it] >> shift) & (NBIN - 1)) : 0xFFFFu;
    uint32_t peers = __match_any_sync(0xffffffffu, d);
    uint32_t rank = __popc(peers & ((1u << lane) - 1u));
    uint32_t dest = 0;
    if (valid) dest = wbase[w][d] + rank;
    __syncwarp();
    if (valid && rank == 0) wbase[w][d] += __popc(peers);
    __syncwarp();
    if (valid) {
      skey[dest] = key[it];
      sval[dest] = vin[i];
    }
  }
  __syncthreads();
  const int nvalid = (int)(n - tile0 < (int64_t)TILE ? n - tile0 : (int64_t)TILE);
#pragma unroll 4
  for (int k = threadIdx.x; k < nvalid; k += SORT_NT) {
    const uint32_t kk = skey[k];
    const uint32_t pos = (uint32_t)k + gdelta[(kk >> shift) & (NBIN - 1)];
    kout[pos] = kk;
    vout[pos] = sval[k];
  }
}

// gather the state into the new order, record slot_of_id for membrane vertices, fill the cell-start table and
// write the pair kernel's records: position relative to the block origin (c & ~1) * edge_q (exact product; the
// subtraction hi - o_c is exact too, so rel carries the full two-float position to ~2^-24), id, concentrations, meta
template <int S>
__global__ void __launch_bounds__(256) k_reorder(const DevParams P, SortedState src, SortedState dst, PairRec rec,
                                                 const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals,
                                                 const uint32_t* __restrict__ rank_cell, int64_t n, uint32_t ncell,
                                                 uint32_t* __restrict__ cell_start, uint32_t* __restrict__ slot_of_id,
                                                 uint32_t* __restrict__ okey, float4* __restrict__ P4ref,
                                                 const uint32_t* __restrict__ gate) {
  TD_GATE(gate);
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t k = keys[i];
  uint32_t from = vals[i];
  float4 p = src.pos[from];
  float4 v = src.vel[from];
  float4 l = src.lo[from];
  uint32_t m = __float_as_uint(l.w);
  dst.pos[i] = p;
  dst.vel[i] = v;
  dst.lo[i] = l;
  float cxv[TD_S - 1];
#pragma unroll
  for (int s = 1; s < TD_S; ++s) cxv[s - 1] = 0.f;
#pragma unroll
  for (int s = 1; s < S; ++s) {
    cxv[s - 1] = src.cx[(int64_t)(s - 1) * n + from];
    dst.cx[(int64_t)(s - 1) * n + i] = cxv[s - 1];
  }
  const uint32_t pc = __ldg(&rank_cell[k]);
  const float ox = (float)(pc & 1022u) * P.edge_q[0], oy = (float)((pc >> 10) & 1022u) * P.edge_q[1],
              oz = (float)((pc >> 20) & 1022u) * P.edge_q[2];  // origin of the 2x2x2 block
  const float4 rel = make_float4(__fadd_rn(__fsub_rn(p.x, ox), l.x), __fadd_rn(__fsub_rn(p.y, oy), l.y),
                                 __fadd_rn(__fsub_rn(p.z, oz), l.z), p.w);
  rec.P4[i] = rel;
  if (okey) { okey[i] = k; P4ref[i] = rel; }  // neighbour-list mode: the binning every later step refers to
  const float4 xr = make_float4(v.w, cxv[0], __uint_as_float(m & 3u), __uint_as_float(m >> 2));
  rec.R8[2 * i] = rel;
  rec.R8[2 * i + 1] = xr;
#pragma unroll
  for (int g = 0; g < td_species_groups(S); ++g)
    rec.Y4[(size_t)g * n + i] = make_float4(cxv[1 + 4 * g], cxv[2 + 4 * g], cxv[3 + 4 * g], cxv[4 + 4 * g]);
  if (m >> 2) slot_of_id[__float_as_uint(p.w)] = (uint32_t)i;
  // cell_start[r] = first slot whose key >= r
  uint32_t kprev = i == 0 ? 0u : keys[i - 1] + 1u;
  if (i == 0 || keys[i - 1] != k)
    for (uint32_t r = kprev; r <= k; ++r) cell_start[r] = (uint32_t)i;
  if (i == n - 1)
    for (uint32_t r = k + 1; r <= ncell; ++r) cell_start[r] = (uint32_t)n;
}
// neighbour-list mode keeps the state on one side: the gathered copy goes back to where the integrator works
template <int S>
__global__ void __launch_bounds__(256) k_copy_state(SortedState src, SortedState dst, int64_t n,
                                                    const uint32_t* __restrict__ gate) {
  TD_GATE(gate);
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  dst.pos[i] = src.pos[i];
  dst.vel[i] = src.vel[i];
  dst.lo[i] = src.lo[i];
#pragma unroll
  for (int s = 1; s < S; ++s) dst.cx[(int64_t)(s - 1) * n + i] = src.cx[(int64_t)(s - 1) * n + i];
}
}  // namespace

int td_sort_passes(int key_bits) { return key_bits <= 0 ? 1 : (key_bits + RB - 1) / RB; }

size_t td_sort_scratch_bytes(int64_t n) {
  int64_t nblk = (n + TILE - 1) / TILE;
  if (nblk < 1) nblk = 1;
  size_t nh = (size_t)nblk * NBIN;
  return (nh + (nh + SCAN_CHUNK - 1) / SCAN_CHUNK + 64) * sizeof(uint32_t);
}

int td_launch_sort(uint32_t* keys[2], uint32_t* vals[2], int64_t n, int key_bits, void* scratch, cudaStream_t st,
                   int* n_launches, const uint32_t* gate) {
  int side = 0;
  if (n == 0) return side;
  int nblk = (int)((n + TILE - 1) / TILE);
  uint32_t* hist = (uint32_t*)scratch;
  const int64_t nh = (int64_t)nblk * NBIN;
  const int nchunk = (int)((nh + SCAN_CHUNK - 1) / SCAN_CHUNK);
  uint32_t* tops = hist + nh;
  int passes = td_sort_passes(key_bits);
  for (int p = 0; p < passes; ++p) {
    int shift = p * RB;
    k_sort_hist<<<nblk, SORT_NT, 0, st>>>(keys[side], n, shift, hist, nblk, gate);
    k_sort_scan<<<nchunk, 1024, 0, st>>>(hist, nh, tops, gate);
    if (nchunk > 1) k_sort_scan_tops<<<1, 1024, 0, st>>>(tops, nchunk, gate);
    k_sort_scatter<<<nblk, SORT_NT, 0, st>>>(keys[side], vals[side], keys[side ^ 1], vals[side ^ 1], n, shift, hist,
                                              nblk, tops, gate);
    side ^= 1;
    if (n_launches) *n_launches += nchunk > 1 ? 4 : 3;
  }
  return side;
}

void td_launch_reorder(const DevParams& P, const SortedState& src, const SortedState& dst, const PairRec& rec,
                       const uint32_t* keys, const uint32_t* vals, const uint32_t* rank_cell, int64_t n,
                       uint32_t ncell, uint32_t* cell_start, uint32_t* slot_of_id, uint32_t* okey, float4* P4ref,
                       const uint32_t* gate, cudaStream_t st) {
  if (n == 0) return;
  int nb = (int)((n + 255) / 256);
  TD_SWITCH_S(P.n_species, k_reorder<S_><<<nb, 256, 0, st>>>(P, src, dst, rec, keys, vals, rank_cell, n, ncell, cell_start,
                                                             slot_of_id, okey, P4ref, gate));
}

void td_launch_copy_state(const DevParams& P, const SortedState& src, const SortedState& dst, int64_t n,
                          const uint32_t* gate, cudaStream_t st) {
  if (n == 0) return;
  int nb = (int)((n + 255) / 256);
  TD_SWITCH_S(P.n_species, k_copy_state<S_><<<nb, 256, 0, st>>>(src, dst, n, gate));
}
