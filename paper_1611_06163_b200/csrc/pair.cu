// pair.cu — row a4 of SURVEY §8(a): the non-bonded tDPD pair kernel.
//   F_i = sum_j [ a w_c - gamma w_R^2 (e.v_ij) + sigma w_R xi / sqrt(dt) ] e_ij      r < r_c   (Eq 2-6)
//   Q_i = sum_j [ -kappa w_cc^{s_c} (C_i - C_j) + sgn_ij m_s sqrt(kappa rho (C_i+C_j)) w_cc^{s_c/2} zeta / sqrt(dt) ]
//                                                                                     r < r_cc  (Eq 7-10)
// Every pair is evaluated on both sides; there are no atomics, so per-particle sums are deterministic.
//
// Design (B200): one CTA owns a brick of 2^k Morton-consecutive cells whose particles are contiguous in the sorted
// order.  The brick's halo (brick +- 1 cell) is staged into shared memory in halo-local x-fastest order, in
// coordinates RELATIVE to the brick origin (periodic images resolved at staging, so the inner loops have no
// minimum-image arithmetic and fp32 differences are exact to ~2^-22).  One thread owns one particle:
//   phase 1 scans the 9 x-runs (3 cells each, contiguous in shared memory) of its stencil and appends the indices of
//           the candidates inside the cutoffs to a private two-ended list in shared memory (front: r < r_c, back:
//           r_c <= r < r_cc), so that
//   phase 2 runs the expensive per-pair work (Philox-4x32-10, Box-Muller, weights) over dense lists instead of
//           under a 14 %-taken branch.
#include "common.cuh"

namespace {

struct PairSmem {
  int* hs;         // [NH + 1] exclusive prefix of halo-cell counts (halo-local x-fastest)
  int* bcs;        // [NCB + 1] brick-cell prefix (Morton rank order) of the brick's own particles
  int* bh;         // [NCB] halo-cell index of each brick cell
  float4* spos;    // [hcap] x', y', z' relative to the brick origin, id bits
  float4* svel;    // [hcap] vx, vy, vz, C_0
  uint32_t* smeta; // [hcap]
  float* scx;      // [(S-1)][hcap]
  uint16_t* list;  // [lcap][NT]
  float* tab;      // type-pair tables
};

__device__ __forceinline__ float td_pow_w(float w, float s) {
  // w in (0,1], s >= 0
  return s == 0.0f ? 1.0f : exp2f(s * __log2f(fmaxf(w, 0.0f)));
}

template <int S, bool RANDFLUX, bool FASTW, bool FORCE>
__device__ __forceinline__ void pair_eval(const DevParams& P, const PairSmem& sm, int hcap, int j, float xi_, float yi,
                                          float zi, const float4& vi, const float* ci, uint32_t idi, uint32_t mi,
                                          uint32_t step, float& fx, float& fy, float& fz, float* q) {
  float4 pj = sm.spos[j];
  float4 vj = sm.svel[j];
  uint32_t mj = sm.smeta[j];
  uint32_t idj = __float_as_uint(pj.w);
  float dx = xi_ - pj.x, dy = yi - pj.y, dz = zi - pj.z;
  float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
  float rinv = rsqrtf(r2);
  float r = r2 * rinv;
  bool excl = P.excl_same && (mi >> 2) != 0u && (mi >> 2) == (mj >> 2);  // R16
  int tt = (int)(mi & 3u) * TD_T + (int)(mj & 3u);
  float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f, g4 = 0.f, g5 = 0.f;
  if (RANDFLUX || FORCE) {
    uint32_t lo = min(idi, idj), hi = max(idi, idj);
    uint32_t x0, x1, x2, x3;
    td_philox(lo, hi, step, 0u, P.key0, P.key1, x0, x1, x2, x3);
    td_box_muller(x0, x1, g0, g1);
    if (RANDFLUX && S >= 2) td_box_muller(x2, x3, g2, g3);
    if (RANDFLUX && S >= 3) {
      td_philox(lo, hi, step, 4u, P.key0, P.key1, x0, x1, x2, x3);
      td_box_muller(x0, x1, g4, g5);
    }
  }
  float keep = excl ? 0.0f : 1.0f;
  if (!FORCE || r2 < P.rcc2) {
    float w = fmaxf(1.0f - r * P.inv_rcc, 0.0f);
    float sgn = idi < idj ? keep : -keep;
#pragma unroll
    for (int s = 0; s < S; ++s) {
      float cj = s == 0 ? vj.w : sm.scx[(s - 1) * hcap + j];
      float kap = sm.tab[(4 + s) * 16 + tt];
      float wdc, wrc;
      if (FASTW) { wdc = w * w; wrc = w; }
      else { wdc = td_pow_w(w, P.s_c[s]); wrc = sqrtf(wdc); }
      float qq = -kap * wdc * (ci[s] - cj) * keep;
      if (RANDFLUX) {
        float zeta = s == 0 ? g1 : s == 1 ? g2 : s == 2 ? g4 : g5;
        float csum = fmaxf(ci[s] + cj, 0.0f);
        qq = fmaf(sgn * zeta * wrc, sqrtf(kap * csum * P.epsc[s]), qq);
      }
      q[s] += qq;
    }
  }
  if (FORCE) {
    float wc = fmaxf(1.0f - r * P.inv_rc, 0.0f);
    float wR, wD;
    if (FASTW) { wR = sqrtf(wc); wD = wc; }
    else { wR = td_pow_w(wc, sm.tab[3 * 16 + tt]); wD = wR * wR; }
    float edv = (dx * (vi.x - vj.x) + dy * (vi.y - vj.y) + dz * (vi.z - vj.z)) * rinv;
    float f = sm.tab[0 * 16 + tt] * wc - sm.tab[1 * 16 + tt] * wD * edv + sm.tab[2 * 16 + tt] * wR * g0;
    f *= rinv * keep;
    fx = fmaf(f, dx, fx);
    fy = fmaf(f, dy, fy);
    fz = fmaf(f, dz, fz);
  }
}

__device__ __forceinline__ PairSmem carve(unsigned char* base, int S, int NH, int NCB, int hcap, int lcap, int NT) {
  PairSmem sm;
  size_t o = 0;
  sm.spos = (float4*)(base + o); o += (size_t)hcap * 16;
  sm.svel = (float4*)(base + o); o += (size_t)hcap * 16;
  sm.smeta = (uint32_t*)(base + o); o += (size_t)hcap * 4;
  sm.scx = (float*)(base + o); o += (size_t)(S - 1) * hcap * 4;
  sm.tab = (float*)(base + o); o += 8 * 16 * 4;
  sm.hs = (int*)(base + o); o += (size_t)(NH + 1) * 4;
  sm.bcs = (int*)(base + o); o += (size_t)(NCB + 1) * 4;
  sm.bh = (int*)(base + o); o += (size_t)NCB * 4;
  o = (o + 15) & ~(size_t)15;
  sm.list = (uint16_t*)(base + o);
  return sm;
}

template <int S, bool RANDFLUX, bool FASTW>
__global__ void __launch_bounds__(256) k_pair(const __grid_constant__ DevParams P, const PairArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NT = blockDim.x, t = threadIdx.x, lane = t & 31, warp = t >> 5, nwarp = NT >> 5;
  const int HX = A.bx + 2, HY = A.by + 2, HZ = A.bz + 2, NH = HX * HY * HZ, NCB = A.bx * A.by * A.bz;
  const int hcap = A.hcap, lcap = A.lcap;
  PairSmem sm = carve(smem_raw, S, NH, NCB, hcap, lcap, NT);
  __shared__ int s_src[6 * 6 * 6];     // first global slot of each halo cell
  __shared__ float s_shift[6 * 6 * 6][3];
  const Brick B = A.bricks[blockIdx.x];

  // ---- type-pair tables
  for (int k = t; k < 16; k += NT) {
    sm.tab[0 * 16 + k] = P.a[k];
    sm.tab[1 * 16 + k] = P.gamma[k];
    sm.tab[2 * 16 + k] = P.sig[k];
    sm.tab[3 * 16 + k] = P.s_R[k];
#pragma unroll
    for (int s = 0; s < TD_S; ++s) sm.tab[(4 + s) * 16 + k] = P.kappa[s][k];
  }
  // ---- halo cells: counts, sources, image shifts
  for (int h = t; h < NH; h += NT) {
    int hx = h % HX, hy = (h / HX) % HY, hz = h / (HX * HY);
    int c[3] = {B.ox + hx - 1, B.oy + hy - 1, B.oz + hz - 1};
    int o[3] = {B.ox, B.oy, B.oz};
    float sh[3];
    bool exists = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      int wimg = 0;
      if (c[a] < 0) { c[a] += P.ncell[a]; wimg = -1; }
      else if (c[a] >= P.ncell[a]) { c[a] -= P.ncell[a]; wimg = 1; }
      // cells beyond a partial brick's extent that would wrap twice cannot occur: ncell >= 3, brick inside the grid
      if (c[a] < 0 || c[a] >= P.ncell[a]) exists = false;
      sh[a] = (float)o[a] * P.cell_edge[a] - (float)wimg * P.box[a];
    }
    uint32_t s0 = 0, s1 = 0;
    if (exists) {
      uint32_t rank = __ldg(&A.cell_rank[(c[2] * P.ncell[1] + c[1]) * P.ncell[0] + c[0]]);
      s0 = __ldg(&A.cell_start[rank]);
      s1 = __ldg(&A.cell_start[rank + 1]);
    }
    s_src[h] = (int)s0;
    sm.hs[h + 1] = (int)(s1 - s0);
    s_shift[h][0] = sh[0]; s_shift[h][1] = sh[1]; s_shift[h][2] = sh[2];
  }
  // ---- brick cells (Morton rank order): own-particle prefix and halo index
  const uint32_t g0 = __ldg(&A.cell_start[B.r0]);
  for (int c = t; c <= (int)B.ncell; c += NT) {
    sm.bcs[c] = (int)(__ldg(&A.cell_start[B.r0 + c]) - g0);
    if (c < (int)B.ncell) {
      uint32_t pc = __ldg(&A.rank_cell[B.r0 + c]);
      int cx = (int)(pc & 1023u) - B.ox, cy = (int)((pc >> 10) & 1023u) - B.oy, cz = (int)(pc >> 20) - B.oz;
      sm.bh[c] = ((cz + 1) * HY + (cy + 1)) * HX + (cx + 1);
    }
  }
  __syncthreads();
  // ---- exclusive scan of halo counts (warp 0, chunks of 32 with carry)
  if (warp == 0) {
    int carry = 0;
    if (lane == 0) sm.hs[0] = 0;
    for (int b0 = 0; b0 < NH; b0 += 32) {
      int h = b0 + lane;
      int v = h < NH ? sm.hs[h + 1] : 0, x = v;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += y;
      }
      if (h < NH) sm.hs[h + 1] = carry + x;
      carry += __shfl_sync(0xffffffffu, x, 31);
    }
  }
  __syncthreads();
  const int nh = sm.hs[NH];
  const int nb = sm.bcs[B.ncell];  // particles owned by this brick
  if (nh > hcap) {                 // cannot stage: report, never write out of bounds
    if (t == 0) atomicOr(A.err, TD_ERR_HALO_OVERFLOW);
    return;
  }
  // ---- stage the halo: one warp per halo cell, coordinates relative to the brick origin
  const int64_t n = A.n;
  for (int h = warp; h < NH; h += nwarp) {
    int d0 = sm.hs[h], cnt = sm.hs[h + 1] - d0, s0 = s_src[h];
    float sx = s_shift[h][0], sy = s_shift[h][1], sz = s_shift[h][2];
    for (int k = lane; k < cnt; k += 32) {
      float4 p = A.st.pos[s0 + k];
      float4 l = A.st.lo[s0 + k];
      p.x = (p.x - sx) + l.x; p.y = (p.y - sy) + l.y; p.z = (p.z - sz) + l.z;
      sm.spos[d0 + k] = p;
      sm.svel[d0 + k] = A.st.vel[s0 + k];
      sm.smeta[d0 + k] = __float_as_uint(l.w);
#pragma unroll
      for (int s = 1; s < S; ++s) sm.scx[(s - 1) * hcap + d0 + k] = A.st.cx[(int64_t)(s - 1) * n + s0 + k];
    }
  }
  __syncthreads();

  // ---- particles of the brick, NT at a time (normally one round)
  for (int p0 = 0; p0 < nb; p0 += NT) {
    const int ip = p0 + t;
    const bool active = ip < nb;
    int self = 0, cbx = 0, cby = 0, cbz = 0;
    if (active) {
      int lo = 0, hi = (int)B.ncell;  // find brick cell c with bcs[c] <= ip < bcs[c+1]
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (sm.bcs[mid] <= ip) lo = mid; else hi = mid;
      }
      int hcell = sm.bh[lo];
      self = sm.hs[hcell] + (ip - sm.bcs[lo]);
      cbx = hcell % HX - 1; cby = (hcell / HX) % HY - 1; cbz = hcell / (HX * HY) - 1;
    }
    float4 pi = sm.spos[active ? self : 0];
    float4 vi = sm.svel[active ? self : 0];
    uint32_t mi = sm.smeta[active ? self : 0];
    uint32_t idi = __float_as_uint(pi.w);
    float ci[S];
    ci[0] = vi.w;
#pragma unroll
    for (int s = 1; s < S; ++s) ci[s] = sm.scx[(s - 1) * hcap + (active ? self : 0)];
    float fx = 0.f, fy = 0.f, fz = 0.f, q[S];
#pragma unroll
    for (int s = 0; s < S; ++s) q[s] = 0.f;
    int nA = 0, nB = 0;

    auto flush = [&]() {
      for (int k = 0; k < nA; ++k)
        pair_eval<S, RANDFLUX, FASTW, true>(P, sm, hcap, sm.list[k * NT + t], pi.x, pi.y, pi.z, vi, ci, idi, mi, A.step,
                                            fx, fy, fz, q);
      for (int k = 0; k < nB; ++k)
        pair_eval<S, RANDFLUX, FASTW, false>(P, sm, hcap, sm.list[(lcap - 1 - k) * NT + t], pi.x, pi.y, pi.z, vi, ci,
                                             idi, mi, A.step, fx, fy, fz, q);
      nA = 0; nB = 0;
    };

    for (int run = 0; run < 9; ++run) {
      int k = 0, kend = 0;
      if (active) {
        int hrow = ((cbz + run / 3) * HY + (cby + run % 3)) * HX + cbx;  // halo cell (cbx-1+1, ...) = first of the run
        k = sm.hs[hrow];
        kend = sm.hs[hrow + 3];
      }
      while (true) {
        int ke = min(kend, k + (lcap - nA - nB));
        for (; k < ke; ++k) {
          float4 pj = sm.spos[k];
          float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
          float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
          if (r2 < P.rcut2 && r2 >= 1e-12f) {  // R22: coincident particles (and self) skipped
            if (r2 < P.rc2) { sm.list[nA * NT + t] = (uint16_t)k; ++nA; }
            else if (r2 < P.rcc2) { sm.list[(lcap - 1 - nB) * NT + t] = (uint16_t)k; ++nB; }
          }
        }
        if (!__any_sync(0xffffffffu, k < kend)) break;
        flush();  // some lane's list is full
      }
    }
    flush();
    if (active) {
      int64_t slot = (int64_t)g0 + ip;
      A.F4[slot] = make_float4(fx, fy, fz, q[0]);
#pragma unroll
      for (int s = 1; s < S; ++s) A.Qx[(int64_t)(s - 1) * n + slot] = q[s];
    }
  }
}

template <int S>
int launch_s(const DevParams& P, const PairArgs& A, int nbricks, int nthreads, size_t smem, cudaStream_t st) {
#define TD_PAIR_GO(RF, FW)                                                                                   \
  do {                                                                                                       \
    auto kf = k_pair<S, RF, FW>;                                                                             \
    cudaError_t e = cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);       \
    if (e != cudaSuccess) return (int)e;                                                                     \
    kf<<<nbricks, nthreads, smem, st>>>(P, A);                                                               \
  } while (0)
  if (P.rand_flux) { if (P.fast_w) TD_PAIR_GO(true, true); else TD_PAIR_GO(true, false); }
  else { if (P.fast_w) TD_PAIR_GO(false, true); else TD_PAIR_GO(false, false); }
#undef TD_PAIR_GO
  return 0;
}
}  // namespace

size_t td_pair_smem_bytes(int S, int bx, int by, int bz, int hcap, int lcap, int nthreads) {
  int NH = (bx + 2) * (by + 2) * (bz + 2), NCB = bx * by * bz;
  size_t o = (size_t)hcap * (16 + 16 + 4 + 4 * (S - 1)) + 8 * 16 * 4 + (size_t)(NH + 1) * 4 + (size_t)(NCB + 1) * 4 +
             (size_t)NCB * 4;
  o = (o + 15) & ~(size_t)15;
  return o + (size_t)lcap * nthreads * 2;
}

int td_launch_pair(const DevParams& P, const PairArgs& A, int nbricks, int nthreads, cudaStream_t st) {
  if (nbricks == 0) return 0;
  size_t smem = td_pair_smem_bytes(P.n_species, A.bx, A.by, A.bz, A.hcap, A.lcap, nthreads);
  switch (P.n_species) {
    case 1: return launch_s<1>(P, A, nbricks, nthreads, smem, st);
    case 2: return launch_s<2>(P, A, nbricks, nthreads, smem, st);
    case 3: return launch_s<3>(P, A, nbricks, nthreads, smem, st);
    default: return launch_s<4>(P, A, nbricks, nthreads, smem, st);
  }
}
