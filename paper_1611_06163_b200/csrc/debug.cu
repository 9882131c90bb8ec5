// debug.cu — read-back and test-support kernels (not on the timed path): scatter of the sorted state back to
// id order for tdpd_get_state, the binning report and exact neighbour census of the bit-exact indexing test
// (DESIGN.md R-bin), and the raw random stream.
#include "common.cuh"

namespace {

// what: 0 pos[n][3], 1 vel[n][3], 2 conc[n][S], 3 force pair+bonded [n][3], 4 flux[n][S], 5 pair force, 6 bonded force
template <int S>
__global__ void __launch_bounds__(256) k_unsort(SortedState st, const float4* __restrict__ F4,
                                                const float* __restrict__ Qx, const float4* __restrict__ Fb, int64_t n,
                                                int what, float* __restrict__ out, int* err, float bx, float by,
                                                float bz) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float4 p = st.pos[i];
  int64_t id = __float_as_uint(p.w);
  float v[S > 3 ? S : 3];
#pragma unroll
  for (int k = 0; k < (S > 3 ? S : 3); ++k) v[k] = 0.f;
  int cnt = 3;
  if (what == 0) {  // hi + lo rounded to fp32, kept inside [0, L): hi = 0 with lo < 0 would round to -1e-9
    float4 l = st.lo[i];
    const float L[3] = {bx, by, bz};
    v[0] = p.x + l.x; v[1] = p.y + l.y; v[2] = p.z + l.z;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (v[a] < 0.0f) v[a] = 0.0f;
      if (v[a] >= L[a]) v[a] = nextafterf(L[a], 0.0f);
    }
  }
  else if (what == 1) { float4 w = st.vel[i]; v[0] = w.x; v[1] = w.y; v[2] = w.z; }
  else if (what == 2) {
    cnt = S;
    v[0] = st.vel[i].w;
#pragma unroll
    for (int s = 1; s < S; ++s) v[s] = st.cx[(int64_t)(s - 1) * n + i];
  } else if (what == 3 || what == 5 || what == 6) {
    if (what != 6) { float4 f = F4[i]; v[0] = f.x; v[1] = f.y; v[2] = f.z; }
    if (what != 5 && (__float_as_uint(st.lo[i].w) >> 2)) { float4 b = Fb[id]; v[0] += b.x; v[1] += b.y; v[2] += b.z; }
  } else {
    cnt = S;
    v[0] = F4[i].w;
#pragma unroll
    for (int s = 1; s < S; ++s) v[s] = Qx[(int64_t)(s - 1) * n + i];
  }
  bool bad = false;
#pragma unroll
  for (int k = 0; k < (S > 3 ? S : 3); ++k)
    if (k < cnt) {
      out[id * cnt + k] = v[k];
      bad |= !isfinite(v[k]);
    }
  if (bad) atomicOr(err, TD_ERR_NONFINITE);
}

// the cells the binning actually used: the sorted key of a slot is the Morton rank of its cell (written by k_integrate,
// td_key_of), rank_cell unpacks it; nothing here re-derives a cell from a position
__global__ void __launch_bounds__(256) k_binning_debug(const DevParams P, SortedState st, int64_t n,
                                                       const uint32_t* __restrict__ keys,
                                                       const uint32_t* __restrict__ rank_cell,
                                                       int32_t* __restrict__ cell_xyz, int32_t* __restrict__ cell_count,
                                                       int32_t* __restrict__ sorted_id) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int64_t id = __float_as_uint(st.pos[i].w);
  const uint32_t pc = rank_cell[keys[i]];
  const int cx = (int)(pc & 1023u), cy = (int)((pc >> 10) & 1023u), cz = (int)(pc >> 20);
  cell_xyz[3 * id] = cx; cell_xyz[3 * id + 1] = cy; cell_xyz[3 * id + 2] = cz;
  if (cell_count) atomicAdd(&cell_count[(cz * P.ncell[1] + cy) * P.ncell[0] + cx], 1);
  if (sorted_id) sorted_id[i] = (int32_t)id;
}

// exact census: differences of fp32 positions in fp64, minimum image, strict cutoffs, through the cell table
__global__ void __launch_bounds__(128) k_census(const DevParams P, SortedState st,
                                                const uint32_t* __restrict__ cell_start,
                                                const uint32_t* __restrict__ cell_rank,
                                                const uint32_t* __restrict__ keys,
                                                const uint32_t* __restrict__ rank_cell, int64_t n,
                                                int32_t* __restrict__ n_rc, int32_t* __restrict__ n_rcc,
                                                uint32_t* __restrict__ xor_rc, uint32_t* __restrict__ xor_rcc) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float4 p = st.pos[i];
  float4 pl = st.lo[i];
  uint32_t mi = __float_as_uint(pl.w);
  int64_t id = __float_as_uint(p.w);
  const uint32_t pc = rank_cell[keys[i]];  // the cell the binning put this slot in
  int c[3] = {(int)(pc & 1023u), (int)((pc >> 10) & 1023u), (int)(pc >> 20)};
  double L[3] = {P.box[0], P.box[1], P.box[2]};
  int a = 0, b = 0;
  uint32_t xa = 0, xb = 0;
  for (int dz = -1; dz <= 1; ++dz)
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        int x = (c[0] + dx + P.ncell[0]) % P.ncell[0], y = (c[1] + dy + P.ncell[1]) % P.ncell[1],
            z = (c[2] + dz + P.ncell[2]) % P.ncell[2];
        uint32_t r = cell_rank[(z * P.ncell[1] + y) * P.ncell[0] + x];
        for (uint32_t k = cell_start[r]; k < cell_start[r + 1]; ++k) {
          if (k == i) continue;
          float4 q = st.pos[k];
          float4 ql = st.lo[k];
          uint32_t mj = __float_as_uint(ql.w);
          if (P.excl_same && (mi >> 2) && (mi >> 2) == (mj >> 2)) continue;
          double d[3] = {((double)p.x + pl.x) - ((double)q.x + ql.x), ((double)p.y + pl.y) - ((double)q.y + ql.y),
                         ((double)p.z + pl.z) - ((double)q.z + ql.z)};
          double r2 = 0.0;
          for (int k2 = 0; k2 < 3; ++k2) {
            d[k2] -= L[k2] * floor(d[k2] / L[k2] + 0.5);
            r2 += d[k2] * d[k2];
          }
          if (r2 < 1e-12) continue;
          double rr = sqrt(r2);
          uint32_t jd = __float_as_uint(q.w);
          if (rr < (double)P.r_c) { ++a; xa ^= jd; }
          if (rr < (double)P.r_cc) { ++b; xb ^= jd; }
        }
      }
  n_rc[id] = a; n_rcc[id] = b; xor_rc[id] = xa; xor_rcc[id] = xb;
}

// overwrite pos / vel / conc of every slot from id-ordered arrays (tdpd_set_state)
template <int S>
__global__ void __launch_bounds__(256) k_set_state(const DevParams P, SortedState st, int64_t n,
                                                   const float* __restrict__ pos, const float* __restrict__ vel,
                                                   const float* __restrict__ conc) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float4 p = st.pos[i];
  int64_t id = __float_as_uint(p.w);
  if (pos) {
    float x[3] = {pos[3 * id], pos[3 * id + 1], pos[3 * id + 2]};
    for (int a = 0; a < 3; ++a) {
      if (x[a] >= P.box[a]) x[a] -= P.box[a];
      if (x[a] < 0.f) { x[a] += P.box[a]; if (x[a] >= P.box[a]) x[a] = 0.f; }
    }
    p.x = x[0]; p.y = x[1]; p.z = x[2];
    st.pos[i] = p;
    float4 l = st.lo[i];
    l.x = l.y = l.z = 0.f;
    st.lo[i] = l;
  }
  if (vel || conc) {
    float4 v = st.vel[i];
    if (vel) { v.x = vel[3 * id]; v.y = vel[3 * id + 1]; v.z = vel[3 * id + 2]; }
    if (conc) {
      v.w = conc[S * id];
#pragma unroll
      for (int s = 1; s < S; ++s) st.cx[(int64_t)(s - 1) * n + i] = conc[S * id + s];
    }
    st.vel[i] = v;
  }
}

__global__ void k_rng_debug(const DevParams P, int64_t n, const int64_t* __restrict__ id_i,
                            const int64_t* __restrict__ id_j, uint32_t step, uint32_t tag, uint32_t* __restrict__ words,
                            float* __restrict__ gauss) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t a = (uint32_t)id_i[i], b = (uint32_t)id_j[i];
  uint32_t x0, x1, x2, x3;
  td_philox(min(a, b), max(a, b), step, tag, P.key0, P.key1, x0, x1, x2, x3);
  if (words) { words[4 * i] = x0; words[4 * i + 1] = x1; words[4 * i + 2] = x2; words[4 * i + 3] = x3; }
  if (gauss) {
    float g0, g1, g2, g3;
    td_box_muller(x0, x1, g0, g1);
    td_box_muller(x2, x3, g2, g3);
    gauss[4 * i] = g0; gauss[4 * i + 1] = g1; gauss[4 * i + 2] = g2; gauss[4 * i + 3] = g3;
  }
}
// Box-Muller of given raw words, through the same device functions the kernels use (u -> 1 series branch included)
__global__ void k_box_muller_debug(int64_t n, const uint32_t* __restrict__ words, float* __restrict__ gauss) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float g0, g1;
  td_box_muller(words[2 * i], words[2 * i + 1], g0, g1);
  gauss[2 * i] = g0; gauss[2 * i + 1] = g1;
}
}  // namespace

void td_launch_box_muller_debug(int64_t n, const uint32_t* words, float* gauss, cudaStream_t st) {
  if (n == 0) return;
  k_box_muller_debug<<<(int)((n + 255) / 256), 256, 0, st>>>(n, words, gauss);
}

void td_launch_unsort(const SortedState& s, const float4* F4, const float* Qx, const float4* Fb, int64_t n,
                      int n_species, int what, float* out, int* err, const float* box, cudaStream_t st) {
  if (n == 0) return;
  int nb = (int)((n + 255) / 256);
  TD_SWITCH_S(n_species, k_unsort<S_><<<nb, 256, 0, st>>>(s, F4, Qx, Fb, n, what, out, err, box[0], box[1], box[2]));
}

void td_launch_binning_debug(const DevParams& P, const SortedState& s, int64_t n, const uint32_t* keys,
                             const uint32_t* rank_cell, int32_t* cell_xyz, int32_t* cell_count, int32_t* sorted_id,
                             cudaStream_t st) {
  if (n == 0) return;
  k_binning_debug<<<(int)((n + 255) / 256), 256, 0, st>>>(P, s, n, keys, rank_cell, cell_xyz, cell_count, sorted_id);
}

void td_launch_census(const DevParams& P, const SortedState& s, const uint32_t* cell_start, const uint32_t* cell_rank,
                      const uint32_t* keys, const uint32_t* rank_cell, int64_t n, int32_t* n_rc, int32_t* n_rcc,
                      uint32_t* xor_rc, uint32_t* xor_rcc, cudaStream_t st) {
  if (n == 0) return;
  k_census<<<(int)((n + 127) / 128), 128, 0, st>>>(P, s, cell_start, cell_rank, keys, rank_cell, n, n_rc, n_rcc, xor_rc,
                                                   xor_rcc);
}

void td_launch_rng_debug(const DevParams& P, int64_t n, const int64_t* id_i, const int64_t* id_j, uint32_t step,
                         uint32_t tag, uint32_t* words, float* gauss, cudaStream_t st) {
  if (n == 0) return;
  k_rng_debug<<<(int)((n + 255) / 256), 256, 0, st>>>(P, n, id_i, id_j, step, tag, words, gauss);
}

void td_launch_set_state(const DevParams& P, const SortedState& s, int64_t n, const float* pos, const float* vel,
                         const float* conc, cudaStream_t st) {
  if (n == 0) return;
  int nb = (int)((n + 255) / 256);
  TD_SWITCH_S(P.n_species, k_set_state<S_><<<nb, 256, 0, st>>>(P, s, n, pos, vel, conc));
}
