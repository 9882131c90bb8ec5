// pair_kernel.cuh — row a4 of SURVEY §8(a): the non-bonded tDPD pair kernel.
//   F_i = sum_j [ a w_c - gamma w_R^2 (e.v_ij) + sigma w_R xi / sqrt(dt) ] e_ij      r < r_c   (Eq 2-6)
//   Q_i = sum_j [ -kappa w_cc^{s_c} (C_i - C_j) + sgn_ij m_s sqrt(kappa rho (C_i+C_j)) w_cc^{s_c/2} zeta / sqrt(dt) ]
//                                                                                     r < r_cc  (Eq 7-10)
// Every pair is evaluated on both sides; there are no atomics, so per-particle sums are deterministic.
//
// Design (B200).  One thread owns one particle of the cell-sorted order; a CTA owns NT consecutive slots, i.e. a
// compact blob of ~NT/13 Morton-consecutive cells.  Nothing is staged: candidate positions are read through L1
// (lanes of one cell read the same address), in coordinates RELATIVE to the origin of their 2x2x2 cell block
// (PairRec::P4), so that the inner loops have no minimum-image arithmetic and fp32 differences are exact to
// ~2^-22 at any box size.
//   prologue  the CTA resolves, for each of its cells, the static neighbour runs (PairArgs::seg_*: the 27
//             neighbour cells merged into ~14 runs of rank-consecutive cells, longest first) against this step's
//             cell table: first slot, particle count, displacement of the run's block origin (periodic image).
//   scan      each thread walks its runs and pushes the hits, branch-free, onto a private two-ended stack of 16-bit
//             entries (run << 11 | offset) in shared memory: front r < min(r_c, r_cc), back the ring up to
//             max(r_c, r_cc).  85 % of the candidates are rejected here for ~14 instructions each.
//   drain     after every run the warp pops the largest multiple of 2 (front) / 4 (back) entries that EVERY lane
//             owns and evaluates them (Philox-4x32-10, Box-Muller, weights), two entries per iteration for
//             instruction-level parallelism, so the expensive loops run with all lanes busy; a full stack or the
//             end of the stencil drains everything.
// Shared memory per thread is ~290 B (24 warps per SM at 80 registers); the first version staged whole halos, ran
// 8 warps per SM and took 4.8x longer.
#pragma once
#include "common.cuh"

#ifndef TD_PAIR_MAXLOC
#define TD_PAIR_MAXLOC 24
#endif
#ifndef TD_PAIR_UNROLL
#define TD_PAIR_UNROLL 8  // measured best of 2 / 4 / 8 / 12 / 16 once the stacks leave no L1: 8 loads in flight per thread
#endif
#ifndef TD_PAIR_ILP
#define TD_PAIR_ILP 2  // list entries evaluated per iteration
#endif
#ifndef TD_PAIR_BA
#define TD_PAIR_BA 2  // drain batch of the front stack (entries; measured best of 2 / 4 / 8)
#endif
#ifndef TD_PAIR_BB
#define TD_PAIR_BB 4  // drain batch of the back stack (measured best of 2 / 4 / 6 / 8 / 16)
#endif
#ifndef TD_PAIR_MINB
#define TD_PAIR_MINB 3
#endif
namespace {

constexpr int MAXLOC = TD_PAIR_MAXLOC;   // cells per table chunk
constexpr int SCAN_UNROLL = TD_PAIR_UNROLL;
constexpr int OFFBITS = 11;  // list entry: neighbour run (0..26) << 11 | offset inside the run
constexpr uint32_t OFFMASK = (1u << OFFBITS) - 1u;

struct PairSmem {
  float4* tso;      // [MAXLOC * 27] first slot (bits), displacement of the neighbour block origin x, y, z
  uint32_t* tcnt;   // [MAXLOC * 27] particles in the neighbour run
  int* tn;          // [MAXLOC] neighbour runs of each local cell
  float* tab;       // [8 * 16] type-pair tables: a, gamma, sigma/sqrt(dt), s_R, kappa[0..3]
  uint16_t* list;   // [lcap][NT]
};

__device__ __forceinline__ float td_pow_w(float w, float s) {
  // w in (0,1], s >= 0
  return s == 0.0f ? 1.0f : exp2f(s * td_lg2_approx(fmaxf(w, 1e-30f)));
}

struct Self {  // the thread's own particle
  float x, y, z;
  float4 v;  // vx, vy, vz, C_0
  float c[TD_S];
  uint32_t id, meta, step;
  int lc27;  // 27 * local cell index
};

// One list entry.  MODE 0: r < min(r_c, r_cc): force and flux; MODE 1: ring with r_cc > r_c: flux only;
// MODE 2: ring with r_c > r_cc: force only.  wgt = 0 turns the entry into a no-op (odd tail of the unrolled loop).
template <int S, bool RANDFLUX, bool FASTW, int MODE>
__device__ __forceinline__ void pair_eval(const DevParams& P, const PairArgs& A, const PairSmem& sm, const Self& me,
                                          uint32_t e, float wgt, float& fx, float& fy, float& fz, float* q) {
  constexpr bool FORCE = MODE != 1, FLUX = MODE != 2;
  const float4 te = sm.tso[me.lc27 + (int)(e >> OFFBITS)];
  const uint32_t j = __float_as_uint(te.x) + (e & OFFMASK);
  const float4 pj = __ldg(&A.rec.P4[j]);
  const float4 xj = __ldg(&A.rec.X4[j]);
  const uint32_t idj = __float_as_uint(pj.w), mj = __float_as_uint(xj.z);
  const float dx = (me.x - te.y) - pj.x, dy = (me.y - te.z) - pj.y, dz = (me.z - te.w) - pj.z;
  const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
  const float rinv = td_rsqrt_approx(fmaxf(r2, 1e-30f));
  const float r = r2 * rinv;
  const bool excl = P.excl_same && (me.meta >> 2) != 0u && (me.meta >> 2) == (mj >> 2);  // R16
  const float keep = (excl || r2 < 1e-12f) ? 0.0f : wgt;                                  // R22
  const int tt = (int)(me.meta & 3u) * TD_T + (int)(mj & 3u);
  float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f, g4 = 0.f, g5 = 0.f;
  if (FORCE || RANDFLUX) {
    const uint32_t lo = min(me.id, idj), hi = max(me.id, idj);
    uint32_t x0, x1, x2, x3;
    td_philox(lo, hi, me.step, 0u, P.key0, P.key1, x0, x1, x2, x3);
    if (FORCE) td_box_muller(x0, x1, g0, g1);  // g0 = xi of the random force
    else td_box_muller_fast(x0, x1, g0, g1);    // flux-only entry: zeta alone
    if (FLUX && RANDFLUX && S >= 2) td_box_muller_fast(x2, x3, g2, g3);
    if (FLUX && RANDFLUX && S >= 3) {
      td_philox(lo, hi, me.step, 4u, P.key0, P.key1, x0, x1, x2, x3);
      td_box_muller_fast(x0, x1, g4, g5);
    }
  }
  if (FLUX) {
    const float w = fmaxf(1.0f - r * P.inv_rcc, 0.0f);
    const float sgn = me.id < idj ? keep : -keep;
#pragma unroll
    for (int s = 0; s < S; ++s) {
      float cj;
      if (s == 0) cj = xj.x;
      else if (s == 1) cj = xj.y;
      else { const float2 y = __ldg(&A.rec.Y2[j]); cj = s == 2 ? y.x : y.y; }
      const float kap = sm.tab[(4 + s) * 16 + tt];
      float wdc, wrc;
      if (FASTW) { wdc = w * w; wrc = w; }
      else { wdc = td_pow_w(w, P.s_c[s]); wrc = td_sqrt_approx(wdc); }
      float qq = -kap * wdc * (me.c[s] - cj) * keep;
      if (RANDFLUX) {
        const float zeta = s == 0 ? g1 : s == 1 ? g2 : s == 2 ? g4 : g5;
        const float csum = fmaxf(me.c[s] + cj, 0.0f);
        qq = fmaf(sgn * zeta * wrc, td_sqrt_approx(kap * csum * P.epsc[s]), qq);
      }
      q[s] += qq;
    }
  }
  if (FORCE) {
    const float4 vj = __ldg(&A.vel[j]);
    // w_c = 1 - r/r_c enters the random force as w_c^s with s < 1 (sqrt for s = 1/2), which is singular at the
    // cutoff: an fp32 error of 1e-7 in r becomes 3e-4 in sqrt(w_c) and 0.03 in the force.  The numerator
    // r_c^2 - r^2 is therefore formed in fp64 from the block-relative coordinates (exact images of the positions
    // whenever the low words are zero, i.e. after load / set_state; rounded to 2^-24 otherwise) and the exact block
    // displacement: w_c = (r_c^2 - r^2) / (r_c (r_c + r)), strict r < r_c as in O2.  14 % of the entries come here.
    const double ex = ((double)me.x - (double)te.y) - (double)pj.x, ey = ((double)me.y - (double)te.z) - (double)pj.y,
                 ez = ((double)me.z - (double)te.w) - (double)pj.z;
    const double rc = (double)P.r_c;
    const float num = (float)(rc * rc - (ex * ex + ey * ey + ez * ez));
    const float wc = fmaxf(num, 0.0f) * td_rcp_approx(P.r_c * (P.r_c + r));
    float wR, wD;
    if (FASTW) { wR = td_sqrt_approx(wc); wD = wc; }
    else { wR = td_pow_w(wc, sm.tab[3 * 16 + tt]); wD = wR * wR; }
    const float edv = (dx * (me.v.x - vj.x) + dy * (me.v.y - vj.y) + dz * (me.v.z - vj.z)) * rinv;
    float f = sm.tab[0 * 16 + tt] * wc - sm.tab[1 * 16 + tt] * wD * edv + sm.tab[2 * 16 + tt] * wR * g0;
    f *= rinv * keep;
    fx = fmaf(f, dx, fx);
    fy = fmaf(f, dy, fy);
    fz = fmaf(f, dz, fz);
  }
}

// evaluates `cnt` entries of one end of the list, two per iteration; entry k of the end lives at base + k * stride
template <int S, bool RANDFLUX, bool FASTW, int MODE>
__device__ __forceinline__ void eval_list(const DevParams& P, const PairArgs& A, const PairSmem& sm, const Self& me,
                                          const uint16_t* base, int stride, int cnt, float& fx, float& fy, float& fz,
                                          float* q) {
#if TD_PAIR_ILP == 1
  for (int k = 0; k < cnt; ++k)
    pair_eval<S, RANDFLUX, FASTW, MODE>(P, A, sm, me, base[k * stride], 1.0f, fx, fy, fz, q);
#else
  for (int k = 0; k < cnt; k += 2) {
    const bool two = k + 1 < cnt;
    const uint32_t e0 = base[k * stride];
    const uint32_t e1 = two ? base[(k + 1) * stride] : e0;
    pair_eval<S, RANDFLUX, FASTW, MODE>(P, A, sm, me, e0, 1.0f, fx, fy, fz, q);
    pair_eval<S, RANDFLUX, FASTW, MODE>(P, A, sm, me, e1, two ? 1.0f : 0.0f, fx, fy, fz, q);
  }
#endif
}

// RING: 1 = r_cc >= r_c (ring entries are flux-only), 2 = r_c > r_cc (ring entries are force-only)
// SPLIT: threads per particle (1, 2, 4 or 16; sub-wave systems): the SPLIT sub-lanes of a particle take every SPLIT-th
// candidate of each run (adjacent addresses), keep private stacks, and their sums are combined by a fixed xor butterfly.
template <int S, bool RANDFLUX, bool FASTW, int RING, int SPLIT>
__global__ void __launch_bounds__(256, TD_PAIR_MINB) k_pair(const __grid_constant__ DevParams P, const PairArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NT = blockDim.x, t = threadIdx.x;
  const int lcap = A.lcap;
  PairSmem sm;
  sm.tso = (float4*)smem_raw;
  sm.tcnt = (uint32_t*)(smem_raw + (size_t)MAXLOC * 27 * 16);
  sm.tab = (float*)(smem_raw + (size_t)MAXLOC * 27 * 20);
  sm.tn = (int*)(smem_raw + (size_t)MAXLOC * 27 * 20 + 8 * 16 * 4);
  sm.list = (uint16_t*)(smem_raw + (size_t)MAXLOC * 27 * 20 + 8 * 16 * 4 + MAXLOC * 4);

  const int64_t n = A.n;
  const int NP = NT / SPLIT, sub = t & (SPLIT - 1);  // particles per CTA, sub-lane of the particle
  const int64_t i0 = (int64_t)blockIdx.x * NP, i = i0 + t / SPLIT;
  const bool active = i < n;
  const int64_t ilast = (i0 + NP < n ? i0 + NP : n) - 1;
  const uint32_t r_first = __ldg(&A.keys[i0]), r_last = __ldg(&A.keys[ilast]);
  const uint32_t ri = active ? __ldg(&A.keys[i]) : 0xFFFFFFFFu;

  Self me;
  {
    const int64_t is = active ? i : i0;
    const float4 p = __ldg(&A.rec.P4[is]);
    const float4 x = __ldg(&A.rec.X4[is]);
    me.x = p.x; me.y = p.y; me.z = p.z;
    me.id = __float_as_uint(p.w);
    me.meta = __float_as_uint(x.z);
    me.v = __ldg(&A.vel[is]);
    me.c[0] = x.x; me.c[1] = x.y; me.c[2] = 0.f; me.c[3] = 0.f;
    if (S > 2) { const float2 y = __ldg(&A.rec.Y2[is]); me.c[2] = y.x; me.c[3] = y.y; }
    me.lc27 = 0;
    me.step = __ldg(A.step_p);
  }
  // ---- type-pair tables
  for (int k = t; k < 16; k += NT) {
    sm.tab[0 * 16 + k] = P.a[k];
    sm.tab[1 * 16 + k] = P.gamma[k];
    sm.tab[2 * 16 + k] = P.sig[k];
    sm.tab[3 * 16 + k] = P.s_R[k];
#pragma unroll
    for (int s = 0; s < TD_S; ++s) sm.tab[(4 + s) * 16 + k] = P.kappa[s][k];
  }
  // list thresholds, inflated by 1e-6 so that no pair inside a cutoff is lost to fp32 rounding of r^2; the
  // weights themselves vanish exactly at the true cutoffs (exact numerator for w_c, clamp for w_cc)
  const float rin2 = fminf(P.rc2, P.rcc2) * 1.000001f, rout2 = P.rcut2 * 1.000001f;
  uint16_t* const lfront = sm.list + t;
  uint16_t* const lback = sm.list + (size_t)(lcap - 1) * NT + t;

  for (uint32_t rb = r_first; rb <= r_last; rb += MAXLOC) {
    const int nloc = (int)min((uint32_t)MAXLOC, r_last - rb + 1u);
    __syncthreads();
    // ---- neighbour runs of the cells rb .. rb + nloc - 1 (static segments + this step's cell table)
    for (int idx = t; idx < nloc * 27; idx += NT) {
      const int lc = idx / 27, k = idx - lc * 27;
      const uint32_t r = rb + lc;
      const uint32_t o0 = __ldg(&A.seg_off[r]), nseg = __ldg(&A.seg_off[r + 1]) - o0;
      if (k == 0) sm.tn[lc] = (int)nseg;
      if ((uint32_t)k < nseg) {
        const uint32_t first = __ldg(&A.seg_first[o0 + k]), meta = __ldg(&A.seg_meta[o0 + k]);
        const uint32_t pc = __ldg(&A.rank_cell[r]), pn = __ldg(&A.rank_cell[first]);
        float off[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          const int ci = (int)((pc >> (10 * a)) & 1022u), cj = (int)((pn >> (10 * a)) & 1022u);  // block coordinates
          const float w = (float)((int)((meta >> (4 + 2 * a)) & 3u) - 1);
          // origin of the neighbour block image - own block origin: both terms exact, their sum too (nearby numbers)
          off[a] = __fadd_rn((float)(cj - ci) * P.edge_q[a], w * P.box[a]);
        }
        const uint32_t s0 = __ldg(&A.cell_start[first]), s1 = __ldg(&A.cell_start[first + (meta & 15u)]);
        uint32_t cnt = s1 - s0;
        if (cnt > OFFMASK) { cnt = OFFMASK; atomicOr(A.err, TD_ERR_CELL_OVERFLOW); }
        sm.tso[idx] = make_float4(__uint_as_float(s0), off[0], off[1], off[2]);
        sm.tcnt[idx] = cnt;
      }
    }
    __syncthreads();
    const bool mine = active && ri >= rb && ri - rb < (uint32_t)nloc;
    me.lc27 = mine ? (int)(ri - rb) * 27 : 0;

    float fx = 0.f, fy = 0.f, fz = 0.f, q[S];
#pragma unroll
    for (int s = 0; s < S; ++s) q[s] = 0.f;
    // two-ended stack: pa grows up from the front, pb down from the back (32-bit shared-memory addresses).
    // Entries are evaluated in warp-uniform batches popped from the tops: after every scanned cell the warp takes
    // the largest multiple of BA (BB) entries that EVERY lane owns, so all lanes run the expensive loops together;
    // a lane whose stack is full, or the end of the stencil, drains everything.
    constexpr int BA = TD_PAIR_BA, BB = TD_PAIR_BB;
    const uint32_t stride = 2u * (uint32_t)NT;
    const int sh = 31 - __clz((int)stride);
    const uint32_t lf32 = (uint32_t)__cvta_generic_to_shared(lfront), lb32 = (uint32_t)__cvta_generic_to_shared(lback);
    uint32_t pa = lf32, pb = lb32;
    const int myn = mine ? sm.tn[me.lc27 / 27] : 0;
    const int clast = __reduce_max_sync(0xffffffffu, myn) - 1;  // warp-uniform number of neighbour runs - 1
    int c = 0;
    float4 te = sm.tso[me.lc27];
    uint32_t e = (uint32_t)sub, ecnt = 0 < myn ? sm.tcnt[me.lc27] : 0u;
    while (true) {
      {
        const float4* __restrict__ src = A.rec.P4 + __float_as_uint(te.x) - ((uint32_t)c << OFFBITS);  // by entry
        const float xs = me.x - te.y, ys = me.y - te.z, zs = me.z - te.w;
        const uint32_t room = (uint32_t)(((int)(pb - pa) >> sh) + 1);  // free entries (pa <= pb + stride always)
        const uint32_t eend = min(ecnt, e + room * SPLIT);
#pragma unroll (SPLIT == 1 ? SCAN_UNROLL : 4)
        for (; e < eend; e += SPLIT) {
          const float4 pj = __ldg(&src[e]);
          const float dx = xs - pj.x, dy = ys - pj.y, dz = zs - pj.z;
          const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
          // branch-free push: front if r2 < rin2, back if rin2 <= r2 < rout2
          asm volatile(
              "{\n\t.reg .pred pin, prg;\n\t"
              "setp.lt.f32 pin, %2, %3;\n\t"
              "setp.lt.and.f32 prg, %2, %4, !pin;\n\t"
              "@pin st.shared.u16 [%0], %5;\n\t"
              "@prg st.shared.u16 [%1], %5;\n\t"
              "@pin add.u32 %0, %0, %6;\n\t"
              "@prg sub.u32 %1, %1, %6;\n\t}"
              : "+r"(pa), "+r"(pb)
              : "f"(r2), "f"(rin2), "f"(rout2), "h"((uint16_t)e), "r"(stride)
              : "memory");
        }
      }
      const bool more = e < ecnt;
      const bool anymore = __any_sync(0xffffffffu, more);
      const int nA = (int)((pa - lf32) >> sh), nB = (int)((lb32 - pb) >> sh);
      int dA, dB;
      if ((!anymore && c >= clast) || __any_sync(0xffffffffu, more && pa > pb)) {
        dA = nA; dB = nB;
      } else {
        const int mA = __reduce_min_sync(0xffffffffu, mine ? nA : 0x7fffffff);
        const int mB = __reduce_min_sync(0xffffffffu, mine ? nB : 0x7fffffff);
        dA = mine ? (mA & ~(BA - 1)) : 0;
        dB = mine ? (mB & ~(BB - 1)) : 0;
      }
      if (__any_sync(0xffffffffu, (dA | dB) != 0)) {
        eval_list<S, RANDFLUX, FASTW, 0>(P, A, sm, me, lfront + (nA - dA) * NT, NT, dA, fx, fy, fz, q);
        eval_list<S, RANDFLUX, FASTW, RING>(P, A, sm, me, lback - (nB - dB) * NT, -NT, dB, fx, fy, fz, q);
        pa -= (uint32_t)dA * stride;
        pb += (uint32_t)dB * stride;
      }
      if (!anymore) {
        if (c >= clast) break;
        ++c;
        te = sm.tso[me.lc27 + c];
        ecnt = ((uint32_t)c << OFFBITS) + (c < myn ? sm.tcnt[me.lc27 + c] : 0u);
        e = ((uint32_t)c << OFFBITS) + (uint32_t)sub;
      }
    }
    if (SPLIT > 1) {
#pragma unroll
      for (int d = 1; d < SPLIT; d <<= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, d);
        fy += __shfl_xor_sync(0xffffffffu, fy, d);
        fz += __shfl_xor_sync(0xffffffffu, fz, d);
#pragma unroll
        for (int s = 0; s < S; ++s) q[s] += __shfl_xor_sync(0xffffffffu, q[s], d);
      }
    }
    if (mine && sub == 0) {
      A.F4[i] = make_float4(fx, fy, fz, q[0]);
#pragma unroll
      for (int s = 1; s < S; ++s) A.Qx[(int64_t)(s - 1) * n + i] = q[s];
    }
  }
}

template <int S, int SPLIT>
int launch_s(const DevParams& P, const PairArgs& A, int nblk, int nthreads, size_t smem, cudaStream_t st) {
#define TD_PAIR_GO(RF, FW, RG)                                                                               \
  do {                                                                                                       \
    auto kf = k_pair<S, RF, FW, RG, SPLIT>;                                                                         \
    cudaError_t e = cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);       \
    if (e != cudaSuccess) return (int)e;                                                                     \
    kf<<<nblk, nthreads, smem, st>>>(P, A);                                                                  \
  } while (0)
  const bool ring1 = P.rcc2 >= P.rc2;
  if (P.rand_flux) {
    if (P.fast_w) { if (ring1) TD_PAIR_GO(true, true, 1); else TD_PAIR_GO(true, true, 2); }
    else { if (ring1) TD_PAIR_GO(true, false, 1); else TD_PAIR_GO(true, false, 2); }
  } else {
    if (P.fast_w) { if (ring1) TD_PAIR_GO(false, true, 1); else TD_PAIR_GO(false, true, 2); }
    else { if (ring1) TD_PAIR_GO(false, false, 1); else TD_PAIR_GO(false, false, 2); }
  }
#undef TD_PAIR_GO
  return 0;
}

template <int SPLIT>
int launch_split(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  if (A.n == 0) return 0;
  const size_t smem = td_pair_smem_bytes(A.lcap, nthreads);
  const int np = nthreads / SPLIT;
  const int nblk = (int)((A.n + np - 1) / np);
  switch (P.n_species) {
    case 1: return launch_s<1, SPLIT>(P, A, nblk, nthreads, smem, st);
    case 2: return launch_s<2, SPLIT>(P, A, nblk, nthreads, smem, st);
    case 3: return launch_s<3, SPLIT>(P, A, nblk, nthreads, smem, st);
    default: return launch_s<4, SPLIT>(P, A, nblk, nthreads, smem, st);
  }
}
}  // namespace
