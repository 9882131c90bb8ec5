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
//             neighbour cells merged into ~14 runs of rank-consecutive cells, longest first) against the cell table
//             of the last binning: first slot, particle count, displacement of the run's block origin (periodic image).
//   candidates  LIST = false: each thread walks its runs (the 27-cell stencil of this step's binning);
//             LIST = true: each thread walks its column of the global
//             neighbour list built by k_build_list at the last binning with cutoff + skin.
//             Hits are pushed, branch-free, onto a private two-ended stack of 16-bit entries (run << 11 | offset) in
//             shared memory: front r < min(r_c, r_cc), back the ring up to max(r_c, r_cc).
//   drain     after every run (chunk of the list) the warp pops the largest multiple of 2 (front) / 4 (back) entries
//             that EVERY lane owns and evaluates them (Philox-4x32-10, Box-Muller, weights), two entries per iteration
//             for instruction-level parallelism, so the expensive loops run with all lanes busy; a full stack or the
//             end of the candidates drains everything.
// Pipe budget of an evaluated entry (measured rates, profiles/r2_peaks.md): 20 IMAD.WIDE at 1.08 / clk / SM and 20
// LOP3 at 2 / clk / SM for Philox, 7-9 MUFU at 0.5 / clk / SM; the evaluation is written to keep the ALU pipe
// (compares, selects, integer adds) and the MUFU count down: exclusion key compare instead of meta arithmetic, dead
// pairs folded into the weights, sqrt(-2 ln u) and sqrt(kappa rho (Ci+Cj)) merged into one square root, packed
// type-pair tables (one LDS.128), self data of the evaluation re-read at every drain instead of held in registers.
#pragma once
#include "common.cuh"

#ifndef TD_PAIR_UNROLL
#define TD_PAIR_UNROLL 8  // measured best of 2 / 4 / 8 / 12 / 16 once the stacks leave no L1: 8 loads in flight per thread
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
#ifndef TD_PAIR_F32X2
#define TD_PAIR_F32X2 1  // packed FADD2 / FMUL2 on the (x, y) pair of a candidate in the stencil scan (-1.3 % kernel time, round 2)
#endif
namespace {

constexpr int MAXLOC = TD_PAIR_MAXLOC;   // cells per table chunk
constexpr int SCAN_UNROLL = TD_PAIR_UNROLL;
constexpr int OFFBITS = 11;  // list entry: neighbour run (0..26) << 11 | offset inside the run
constexpr uint32_t OFFMASK = (1u << OFFBITS) - 1u;
__host__ __device__ constexpr int td_ngroups(int S) { return S <= 2 ? 0 : (S - 2 + 3) / 4; }  // float4 groups of the species beyond C_1

struct PairSmem {
  float4* tso;      // [MAXLOC * 27] first slot (bits), displacement of the neighbour block origin x, y, z
  uint32_t* tcnt;   // [MAXLOC * 27] particles in the neighbour run
  int* tn;          // [MAXLOC] neighbour runs of each local cell
  float4* tabF;     // [16] type-pair table: a, gamma, sigma/sqrt(dt), s_R
  float* tabK;      // [TD_S][16] kappa per species and type pair
  uint16_t* list;   // [lcap][NT]
};

__device__ __forceinline__ float td_pow_w(float w, float s) {
  // w in [0,1], s >= 0; 0 at w = 0 whatever s (a weight beyond its cutoff, also for s = 0)
  return w > 0.0f ? exp2f(s * td_lg2_approx(w)) : 0.0f;
}

// The thread's own particle.  x, y, z and lc27 live through the candidate loops; the rest is needed by the evaluation
// only and is re-read (L1) at the start of every drain, so that it holds no registers while candidates are scanned.
template <int S>
struct Self {
  float x, y, z;
  int lc27;       // 27 * local cell index
  float4 v;  // vx, vy, vz, C_0
  float c[S];
  uint32_t id, step;
  uint32_t exq;   // exclusion key to compare with a candidate's X4.w: own membrane + 1, or ~0 (never equal) (R16)
  int t4;         // type * TD_T
};

// fp32 word -> f = 1.m in [1, 2) with m = x >> 9; the uniform of DESIGN.md R-RNG is u = f - (1 - 2^-24)
__device__ __forceinline__ float td_f12(uint32_t x) { return __uint_as_float((x >> 9) | 0x3f800000u); }
constexpr float TD_C0 = 0.99999994039535522f;          // 1 - 2^-24
constexpr float TD_TWO_PI = 6.283185307179586f;
constexpr float TD_ANG0 = -6.2831849326109f;           // -2 pi (1 - 2^-24)
constexpr float TD_M2LN2 = -1.3862943611198906f;       // -2 ln 2
// angle 2 pi u of the word xb in one FMA
__device__ __forceinline__ float td_angle(uint32_t xb) { return fmaf(td_f12(xb), TD_TWO_PI, TD_ANG0); }

// One list entry.  MODE 0: r < min(r_c, r_cc): force and flux; MODE 1: ring with r_cc > r_c: flux only;
// MODE 2: ring with r_c > r_cc: force only.  live = false turns the entry into a no-op (odd tail of the unrolled loop).
template <int S, bool RANDFLUX, bool FASTW, int MODE>
__device__ __forceinline__ void pair_eval(const DevParams& P, const PairArgs& A, const PairSmem& sm, const Self<S>& me,
                                          uint32_t e, bool live, float& fx, float& fy, float& fz, float* q) {
  constexpr bool FORCE = MODE != 1, FLUX = MODE != 2;
  constexpr int NG = td_ngroups(S);
  const float4 te = sm.tso[me.lc27 + (int)(e >> OFFBITS)];
  const uint32_t j = __float_as_uint(te.x) + (e & OFFMASK);
  float4 pj, xj;  // one 256-bit load of the neighbour's record (position + id, concentrations + type + exclusion key)
  asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
      : "=f"(pj.x), "=f"(pj.y), "=f"(pj.z), "=f"(pj.w), "=f"(xj.x), "=f"(xj.y), "=f"(xj.z), "=f"(xj.w)
      : "l"(A.rec.R8 + 2 * (size_t)j));
  const uint32_t idj = __float_as_uint(pj.w);
  const float dx = (me.x - te.y) - pj.x, dy = (me.y - te.z) - pj.y, dz = (me.z - te.w) - pj.z;
  const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
  const float rinv = td_rsqrt_approx(fmaxf(r2, 1e-30f));
  const float r = r2 * rinv;
  // dead pairs: same membrane (R16), coincident particles (R22), the padding entry of an odd tail
  const bool dead = __float_as_uint(xj.w) == me.exq || r2 < 1e-12f || !live;
  const int tt = me.t4 + (int)__float_as_uint(xj.z);
  uint32_t x0 = 0, x1 = 0, x2 = 0, x3 = 0;
  const uint32_t lo = min(me.id, idj), hi = max(me.id, idj);
  if (FORCE || RANDFLUX) td_philox(lo, hi, me.step, 0u, P.key0, P.key1, x0, x1, x2, x3);
  const float l0 = (FORCE || RANDFLUX) ? td_lg2_approx(td_f12(x0) - TD_C0) : 0.0f;  // lg2 u(x0) <= 0
  if (FLUX) {
    float w = fmaxf(fmaf(-r, P.inv_rcc, 1.0f), 0.0f);
    w = dead ? 0.0f : w;
    const bool up = me.id < idj;  // sgn_ij = +1 if id_i < id_j (R5)
    float4 yj[NG > 0 ? NG : 1];
#pragma unroll
    for (int g = 0; g < NG; ++g) yj[g] = __ldg(&A.rec.Y4[(size_t)g * A.n + j]);
    // random words of the species: 0: (x0,x1) sin; 1: (x2,x3) cos; 2+4g..5+4g: tag 4+g, (x0,x1) cos, sin, (x2,x3) cos, sin
    float lg[1 + NG * 2 + 1], tr[S];
    if (RANDFLUX) {
      lg[0] = l0;
      tr[0] = td_sin_approx(td_angle(x1));
      if (S >= 2) {
        lg[1] = td_lg2_approx(td_f12(x2) - TD_C0);
        tr[1] = td_cos_approx(td_angle(x3));
      }
#pragma unroll
      for (int g = 0; g < NG; ++g) {
        uint32_t y0, y1, y2, y3;
        td_philox(lo, hi, me.step, 4u + g, P.key0, P.key1, y0, y1, y2, y3);
        lg[2 + 2 * g] = td_lg2_approx(td_f12(y0) - TD_C0);
        const float a01 = td_angle(y1);
        tr[2 + 4 * g] = td_cos_approx(a01);
        if (3 + 4 * g < S) tr[3 + 4 * g] = td_sin_approx(a01);
        if (4 + 4 * g < S) {
          lg[3 + 2 * g] = td_lg2_approx(td_f12(y2) - TD_C0);
          const float a23 = td_angle(y3);
          tr[4 + 4 * g] = td_cos_approx(a23);
          if (5 + 4 * g < S) tr[5 + 4 * g] = td_sin_approx(a23);
        }
      }
    }
    float wdc_f = w * w, sgnw_f = up ? w : -w;  // FASTW: s_c = 2 for every species
#pragma unroll
    for (int s = 0; s < S; ++s) {
      float cj;
      if (s == 0) cj = xj.x;
      else if (s == 1) cj = xj.y;
      else { const float4 y = yj[(s - 2) / 4]; const int k = (s - 2) & 3; cj = k == 0 ? y.x : k == 1 ? y.y : k == 2 ? y.z : y.w; }
      const float kap = sm.tabK[s * 16 + tt];
      float wdc, sgnw;
      if (FASTW) { wdc = wdc_f; sgnw = sgnw_f; }
      else { wdc = td_pow_w(w, P.s_c[s]); const float wrc = td_sqrt_approx(wdc); sgnw = up ? wrc : -wrc; }
      q[s] = fmaf(-(kap * wdc), me.c[s] - cj, q[s]);
      if (RANDFLUX) {
        // zeta sqrt(kappa rho m_s^2 (Ci+Cj) / dt) = trig sqrt(-2 ln u kappa (Ci+Cj) epsc): one square root (Eq 9-10)
        const float lgs = s == 0 ? lg[0] : s == 1 ? lg[1] : lg[2 + 2 * ((s - 2) / 4) + (((s - 2) & 3) >> 1)];
        const float csum = fmaxf(me.c[s] + cj, 0.0f);
        const float rt = td_sqrt_approx((kap * csum) * (lgs * P.epsc2[s]));
        q[s] = fmaf(rt * tr[s], sgnw, q[s]);
      }
    }
  }
  if (FORCE) {
    const float4 vj = __ldg(&A.vel[j]);
    const float4 tf = sm.tabF[tt];  // a, gamma, sigma / sqrt(dt), s_R
    // w_c = 1 - r/r_c enters the random force as w_c^s with s < 1 (sqrt for s = 1/2), which is singular at the
    // cutoff: an fp32 error of 1e-7 in r becomes 3e-4 in sqrt(w_c) and 0.03 in the force.  The numerator
    // r_c^2 - r^2 is therefore formed in fp64 from the block-relative coordinates (exact images of the positions
    // whenever the low words are zero, i.e. after load / set_state; rounded to 2^-24 otherwise) and the exact block
    // displacement: w_c = (r_c^2 - r^2) / (r_c (r_c + r)), strict r < r_c as in O2.  14 % of the entries come here.
    // (Taking this path only where the fp32 w_c is small was measured in round 2: the branch splits the two
    // interleaved entries and costs 160 B of spills at 80 registers.)
    float wc;
    {
      const double ex = ((double)me.x - (double)te.y) - (double)pj.x, ey = ((double)me.y - (double)te.z) - (double)pj.y,
                   ez = ((double)me.z - (double)te.w) - (double)pj.z;
      const double rc = (double)P.r_c;
      const float num = (float)(rc * rc - (ex * ex + ey * ey + ez * ez));
      wc = fmaxf(num, 0.0f) * td_rcp_approx(P.r_c * (P.r_c + r));
    }
    float wR, wD;
    if (FASTW) { wR = td_sqrt_approx(wc); wD = wc; }
    else { wR = td_pow_w(wc, tf.w); wD = wR * wR; }
    // xi = R cos(2 pi u1), R = sqrt(-2 ln u0); near u0 = 1 (R -> 0) lg2.approx is not accurate enough: series (td_bm_radius)
    const float R0 = td_bm_radius_l(td_f12(x0) - TD_C0, l0);
    const float g0 = R0 * td_cos_approx(td_angle(x1));
    const float edv = (dx * (me.v.x - vj.x) + dy * (me.v.y - vj.y) + dz * (me.v.z - vj.z)) * rinv;
    float f = fmaf(tf.z * wR, g0, fmaf(-(tf.y * wD), edv, tf.x * wc));
    f *= dead ? 0.0f : rinv;
    fx = fmaf(f, dx, fx);
    fy = fmaf(f, dy, fy);
    fz = fmaf(f, dz, fz);
  }
}

// evaluates `cnt` entries of one end of the list, two per iteration; entry k of the end lives at base + k * stride
template <int S, bool RANDFLUX, bool FASTW, int MODE>
__device__ __forceinline__ void eval_list(const DevParams& P, const PairArgs& A, const PairSmem& sm, const Self<S>& me,
                                          const uint16_t* base, int stride, int cnt, float& fx, float& fy, float& fz,
                                          float* q) {
  if (A.census) {
    // test support (tdpd_debug_pair_census): instead of evaluating, count the entries the REAL candidate loops put on
    // this end of the stack and XOR the ids behind them (same run tables, same thresholds, same dead-pair rule)
    uint32_t c = 0, x = 0;
    for (int k = 0; k < cnt; ++k) {
      const uint32_t e = base[k * stride];
      const float4 te = sm.tso[me.lc27 + (int)(e >> OFFBITS)];
      const uint32_t j = __float_as_uint(te.x) + (e & OFFMASK);
      const float4 pj = __ldg(&A.rec.R8[2 * (size_t)j]), xj = __ldg(&A.rec.R8[2 * (size_t)j + 1]);
      const float dx = (me.x - te.y) - pj.x, dy = (me.y - te.z) - pj.y, dz = (me.z - te.w) - pj.z;
      if (__float_as_uint(xj.w) == me.exq || fmaf(dz, dz, fmaf(dy, dy, dx * dx)) < 1e-12f) continue;
      ++c; x ^= __float_as_uint(pj.w);
    }
    if (cnt > 0) {
      uint32_t* out = A.census + (size_t)(MODE == 0 ? 0 : 2) * (size_t)A.n + me.id;
      atomicAdd(out, c);
      atomicXor(out + A.n, x);
    }
    return;
  }
  for (int k = 0; k < cnt; k += 2) {
    const bool two = k + 1 < cnt;
    const uint32_t e0 = base[k * stride];
    const uint32_t e1 = two ? base[(k + 1) * stride] : e0;
    pair_eval<S, RANDFLUX, FASTW, MODE>(P, A, sm, me, e0, true, fx, fy, fz, q);
    pair_eval<S, RANDFLUX, FASTW, MODE>(P, A, sm, me, e1, two, fx, fy, fz, q);
  }
}

__device__ __forceinline__ PairSmem td_pair_carve(unsigned char* smem_raw) {
  PairSmem sm;
  sm.tso = (float4*)smem_raw;
  sm.tabF = (float4*)(smem_raw + (size_t)MAXLOC * 27 * 16);
  sm.tcnt = (uint32_t*)(smem_raw + (size_t)MAXLOC * 27 * 16 + 16 * 16);
  sm.tabK = (float*)(smem_raw + (size_t)MAXLOC * 27 * 20 + 16 * 16);
  sm.tn = (int*)(smem_raw + (size_t)MAXLOC * 27 * 20 + 16 * 16 + (size_t)TD_S * 16 * 4);
  sm.list = (uint16_t*)(smem_raw + td_pair_table_bytes());
  return sm;
}

// neighbour runs of the cells rb .. rb + nloc - 1 (static segments + the cell table of the last binning)
__device__ __forceinline__ void td_pair_fill_table(const DevParams& P, const PairArgs& A, const PairSmem& sm, uint32_t rb,
                                                   int nloc, int t, int NT) {
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
}

// the evaluation-time part of Self
template <int S>
__device__ __forceinline__ void td_pair_load_self(const DevParams& P, const PairArgs& A, int64_t is, Self<S>& me) {
  constexpr int NG = td_ngroups(S);
  const float4 x = __ldg(&A.rec.R8[2 * is + 1]);
  me.id = __float_as_uint(__ldg(&A.rec.P4[is].w));
  me.t4 = (int)__float_as_uint(x.z) * TD_T;
  const uint32_t k = __float_as_uint(x.w);
  me.exq = (k && P.excl_same) ? k : 0xFFFFFFFFu;
  me.v = __ldg(&A.vel[is]);
  me.c[0] = x.x;
  if (S >= 2) me.c[1] = x.y;
#pragma unroll
  for (int g = 0; g < NG; ++g) {
    const float4 y = __ldg(&A.rec.Y4[(size_t)g * A.n + is]);
    if (2 + 4 * g < S) me.c[2 + 4 * g] = y.x;
    if (3 + 4 * g < S) me.c[3 + 4 * g] = y.y;
    if (4 + 4 * g < S) me.c[4 + 4 * g] = y.z;
    if (5 + 4 * g < S) me.c[5 + 4 * g] = y.w;
  }
  me.step = __ldg(A.step_p);
}

// branch-free two-ended push: front if r2 < rin2, back if rin2 <= r2 < rout2
__device__ __forceinline__ void td_push2(uint32_t& pa, uint32_t& pb, float r2, float rin2, float rout2, uint32_t e,
                                         uint32_t stride) {
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

// RING: 1 = r_cc >= r_c (ring entries are flux-only), 2 = r_c > r_cc (ring entries are force-only)
// SPLIT: threads per particle (1, 2, 4 or 16; sub-wave systems): the SPLIT sub-lanes of a particle take every SPLIT-th
// candidate of each run (adjacent addresses), keep private stacks, and their sums are combined by a fixed xor butterfly.
// LIST: candidates come from the global neighbour list (SPLIT == 1 only) instead of the 27-cell stencil.
template <int S, bool RANDFLUX, bool FASTW, int RING, int SPLIT, bool LIST>
__global__ void __launch_bounds__(256, (S >= 6 ? 2 : TD_PAIR_MINB)) k_pair(const __grid_constant__ DevParams P, const PairArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NT = blockDim.x, t = threadIdx.x;
  const int lcap = A.lcap;
  const PairSmem sm = td_pair_carve(smem_raw);

  const int64_t n = A.n;
  const int NP = NT / SPLIT, sub = t & (SPLIT - 1);  // particles per CTA, sub-lane of the particle
  const int64_t i0 = (int64_t)blockIdx.x * NP, i = i0 + t / SPLIT;
  const bool active = i < n;
  const int64_t ilast = (i0 + NP < n ? i0 + NP : n) - 1;
  const uint32_t r_first = __ldg(&A.keys[i0]), r_last = __ldg(&A.keys[ilast]);
  const uint32_t ri = active ? __ldg(&A.keys[i]) : 0xFFFFFFFFu;

  Self<S> me;
  const int64_t is = active ? i : i0;
  {
    const float4 p = __ldg(&A.rec.P4[is]);
    me.x = p.x; me.y = p.y; me.z = p.z;
    me.lc27 = 0;
  }
  // ---- type-pair tables
  for (int k = t; k < 16; k += NT) {
    sm.tabF[k] = make_float4(P.a[k], P.gamma[k], P.sig[k], P.s_R[k]);
#pragma unroll
    for (int s = 0; s < TD_S; ++s) sm.tabK[s * 16 + k] = P.kappa[s][k];
  }
  // list thresholds, inflated by 1e-6 so that no pair inside a cutoff is lost to fp32 rounding of r^2; the
  // weights themselves vanish exactly at the true cutoffs (exact numerator for w_c, clamp for w_cc)
  const float rin2 = fminf(P.rc2, P.rcc2) * 1.000001f, rout2 = P.rcut2 * 1.000001f;
  uint16_t* const lfront = sm.list + t;
  uint16_t* const lback = sm.list + (size_t)(lcap - 1) * NT + t;
  // LIST: this thread's column of the global neighbour list (tiles of 256 slots, [tile][entry][lane])
  const uint16_t* gcol = nullptr;
  uint32_t gcnt = 0;
  if (LIST) {
    gcol = A.nlist + ((size_t)(i0 >> 8) * A.nl_cap) * 256 + (size_t)(i - i0);
    gcnt = active ? __ldg(&A.nl_cnt[i]) : 0u;
  }

  for (uint32_t rb = r_first; rb <= r_last; rb += MAXLOC) {
    const int nloc = (int)min((uint32_t)MAXLOC, r_last - rb + 1u);
    __syncthreads();
    td_pair_fill_table(P, A, sm, rb, nloc, t, NT);
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
    // warp-uniform number of candidate chunks - 1: neighbour runs (scan) or LCHUNK-entry pieces of the list column
    constexpr uint32_t LCHUNK = 32;
    const int clast = LIST ? (int)((__reduce_max_sync(0xffffffffu, mine ? gcnt : 0u) + LCHUNK - 1) / LCHUNK) - 1
                           : __reduce_max_sync(0xffffffffu, myn) - 1;
    int c = 0;
    float4 te = sm.tso[me.lc27];
    uint32_t e = LIST ? 0u : (uint32_t)sub;
    uint32_t ecnt = LIST ? (mine ? min(gcnt, LCHUNK) : 0u) : (0 < myn ? sm.tcnt[me.lc27] : 0u);
    while (true) {
      const uint32_t room = (uint32_t)(((int)(pb - pa) >> sh) + 1);  // free entries (pa <= pb + stride always)
      if (LIST) {
        const uint32_t eend = min(ecnt, e + room);
#pragma unroll 4
        for (; e < eend; ++e) {
          const uint32_t le = gcol[(size_t)e * 256];
          const float4 tl = sm.tso[me.lc27 + (int)(le >> OFFBITS)];
          const float4 pj = __ldg(&A.rec.P4[__float_as_uint(tl.x) + (le & OFFMASK)]);
          const float dx = (me.x - tl.y) - pj.x, dy = (me.y - tl.z) - pj.y, dz = (me.z - tl.w) - pj.z;
          const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
          td_push2(pa, pb, r2, rin2, rout2, le, stride);
        }
      } else {
        const float4* __restrict__ src = A.rec.P4 + __float_as_uint(te.x) - ((uint32_t)c << OFFBITS);  // by entry
        const float xs = me.x - te.y, ys = me.y - te.z, zs = me.z - te.w;
        const uint32_t eend = min(ecnt, e + room * SPLIT);
#pragma unroll (SPLIT == 1 ? SCAN_UNROLL : 4)
        for (; e < eend; e += SPLIT) {
          const float4 pj = __ldg(&src[e]);
#if TD_PAIR_F32X2
          // x and y of a candidate arrive in an aligned register pair: their difference and square go through the packed
          // FP32 pipe of sm_100 (FADD2 / FMUL2 in SASS), 5 instead of 6 instructions per distance test
          float qx, qy;
          asm("{.reg .b64 s, p, d;\n\tmov.b64 s, {%2, %3};\n\tmov.b64 p, {%4, %5};\n\t"
              "sub.rn.f32x2 d, s, p;\n\tmul.rn.f32x2 d, d, d;\n\tmov.b64 {%0, %1}, d;\n\t}"
              : "=f"(qx), "=f"(qy) : "f"(xs), "f"(ys), "f"(pj.x), "f"(pj.y));
          const float dz = zs - pj.z;
          const float r2 = fmaf(dz, dz, qx) + qy;
#else
          const float dx = xs - pj.x, dy = ys - pj.y, dz = zs - pj.z;
          const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
#endif
          td_push2(pa, pb, r2, rin2, rout2, e, stride);
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
        td_pair_load_self<S>(P, A, is, me);
        eval_list<S, RANDFLUX, FASTW, 0>(P, A, sm, me, lfront + (nA - dA) * NT, NT, dA, fx, fy, fz, q);
        eval_list<S, RANDFLUX, FASTW, RING>(P, A, sm, me, lback - (nB - dB) * NT, -NT, dB, fx, fy, fz, q);
        pa -= (uint32_t)dA * stride;
        pb += (uint32_t)dB * stride;
      }
      if (!anymore) {
        if (c >= clast) break;
        ++c;
        if (LIST) {
          ecnt = mine ? min(gcnt, (uint32_t)(c + 1) * LCHUNK) : 0u;
        } else {
          te = sm.tso[me.lc27 + c];
          ecnt = ((uint32_t)c << OFFBITS) + (c < myn ? sm.tcnt[me.lc27 + c] : 0u);
          e = ((uint32_t)c << OFFBITS) + (uint32_t)sub;
        }
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
      if (P.has_source) {  // Q^S_i of Eq 7: external source and first-order reaction by species and type
        td_pair_load_self<S>(P, A, i, me);
        const int ty = me.t4 / TD_T;
#pragma unroll
        for (int s = 0; s < S; ++s)
          if (s < P.n_species) q[s] += P.src[s][ty] - P.dec[s][ty] * me.c[s];
      }
      A.F4[i] = make_float4(fx, fy, fz, q[0]);
#pragma unroll
      for (int s = 1; s < S; ++s)
        if (s < P.n_species) A.Qx[(int64_t)(s - 1) * n + i] = q[s];
    }
  }
}


template <int S, int SPLIT, bool LIST>
int launch_s(const DevParams& P, const PairArgs& A, int nblk, int nthreads, size_t smem, cudaStream_t st) {
#define TD_PAIR_GO(RF, FW, RG)                                                                               \
  do {                                                                                                       \
    auto kf = k_pair<S, RF, FW, RG, SPLIT, LIST>;                                                            \
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

// species counts are rounded up to the compiled set {1, 2, 4, 6, 10}: a padded species has kappa = 0 and C = 0, so
// its flux is exactly zero and is never stored
template <int SPLIT, bool LIST>
int launch_split(const DevParams& P, const PairArgs& A, int nthreads, cudaStream_t st) {
  if (A.n == 0) return 0;
  const size_t smem = td_pair_smem_bytes(A.lcap, nthreads);
  const int np = nthreads / SPLIT;
  const int nblk = (int)((A.n + np - 1) / np);
  switch (td_species_padded(P.n_species)) {
    case 1: return launch_s<1, SPLIT, LIST>(P, A, nblk, nthreads, smem, st);
    case 2: return launch_s<2, SPLIT, LIST>(P, A, nblk, nthreads, smem, st);
    case 4: return launch_s<4, SPLIT, LIST>(P, A, nblk, nthreads, smem, st);
    case 6: return launch_s<6, SPLIT, LIST>(P, A, nblk, nthreads, smem, st);
    default: return launch_s<10, SPLIT, LIST>(P, A, nblk, nthreads, smem, st);
  }
}
}  // namespace
