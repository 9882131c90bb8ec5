// integrate.cu — rows a1 and a9 of SURVEY §8(a): velocity-Verlet half-kicks of velocity and concentration, drift,
// periodic wrap and the cell hash, fused (R21; BASELINE north_star (4) — the paper does not describe
// its integrator).  Runs in the cell-sorted order of the previous binning.
#include "common.cuh"

// cell coordinate along one axis (DESIGN.md R-bin): c = min(n-1, floor(x * inv)), one rounded fp32 multiply
__device__ __forceinline__ int td_cell_axis(float x, float inv, int n) {
  int c = (int)floorf(__fmul_rn(x, inv));
  c = c > n - 1 ? n - 1 : c;
  return c < 0 ? 0 : c;
}

// drift of one coordinate held as a two-float number (hi + lo): x += dt v, then the periodic wrap, with every
// rounding error carried in lo, so that the trajectory is integrated to ~2^-46 relative while all force
// arithmetic stays fp32.  (Positions rounded to fp32 each step would lose ulp(L)/2 per step: 4e-6 at L = 128.)
__device__ __forceinline__ void td_drift(float& hi, float& lo, float dt, float v, float L) {
  float s = fmaf(dt, v, lo);
  float h = __fadd_rn(hi, s);
  float bb = __fsub_rn(h, hi);
  float e = __fadd_rn(__fsub_rn(hi, __fsub_rn(h, bb)), __fsub_rn(s, bb));  // TwoSum error term
  if (h >= L) {
    h = __fsub_rn(h, L);  // exact for h in [L, 2L)
  } else if (h < 0.0f) {
    float h2 = __fadd_rn(h, L);
    float b2 = __fsub_rn(h2, h);
    e = __fadd_rn(e, __fadd_rn(__fsub_rn(h, __fsub_rn(h2, b2)), __fsub_rn(L, b2)));
    h = h2;
    if (h >= L) h = 0.0f;  // image of a tiny negative number: L == 0, the remainder stays in lo
  }
  hi = h;
  lo = e;
}

__device__ __forceinline__ uint32_t td_key_of(const DevParams& P, float x, float y, float z,
                                              const uint32_t* __restrict__ cell_rank) {
  int cx = td_cell_axis(x, P.cell_inv[0], P.ncell[0]);
  int cy = td_cell_axis(y, P.cell_inv[1], P.ncell[1]);
  int cz = td_cell_axis(z, P.cell_inv[2], P.ncell[2]);
  return __ldg(&cell_rank[(cz * P.ncell[1] + cy) * P.ncell[0] + cx]);
}

// body acceleration sign at the force-evaluation position (R14)
__device__ __forceinline__ float td_body_sign(const DevParams& P, float z) {
  if (P.body_mode == 1) return 1.0f;
  if (P.body_mode == 2) return z < P.half_box_z ? 1.0f : -1.0f;
  return 0.0f;
}

template <int S>
__device__ __forceinline__ void td_half_kick(const DevParams& P, float4& p, float4& v, float* cx_val,
                                             const float4* __restrict__ F4, const float* __restrict__ Qx,
                                             const float4* __restrict__ Fb, uint32_t meta, int64_t i, int64_t n) {
  float4 f = F4[i];
  if (meta >> 2) {  // membrane vertex: add the bonded force (stored by id)
    float4 b = Fb[__float_as_uint(p.w)];
    f.x += b.x; f.y += b.y; f.z += b.z;
  }
  float sg = td_body_sign(P, p.z);
  float h = P.half_dt;
  v.x = fmaf(h, f.x + sg * P.body[0], v.x);
  v.y = fmaf(h, f.y + sg * P.body[1], v.y);
  v.z = fmaf(h, f.z + sg * P.body[2], v.z);
  v.w = fmaf(h, f.w, v.w);
#pragma unroll
  for (int s = 1; s < S; ++s) cx_val[s - 1] = fmaf(h, Qx[(int64_t)(s - 1) * n + i], cx_val[s - 1]);
}

// mode: 0 = keys only (initial binning), 1 = opening half-kick + drift + wrap + key,
//       2 = closing half-kick of the previous step, then mode 1, 3 = closing half-kick only
// LISTM (neighbour list reused between binnings): the particles keep the slots of the last
// binning, so the kernel also refreshes the pair kernel's records in place (position relative to the block origin
// of the cell the particle was binned into, unwrapped through the periodic boundary; concentrations) and takes the
// maximum displacement since that binning, which decides on the device whether this step re-bins (k_list_decide).
template <int S, bool LISTM>
__global__ void __launch_bounds__(256) k_integrate(const DevParams P, SortedState st, const float4* __restrict__ F4,
                                                   const float* __restrict__ Qx, const float4* __restrict__ Fb,
                                                   int64_t n, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                                   const uint32_t* __restrict__ cell_rank, int mode,
                                                   uint32_t* __restrict__ ctl, ListRefresh LR) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.0f;
  if (i < n) {
    if (i == 0 && ctl) {
      ctl[TD_CTL_STEP] += 1u;   // the force evaluation that follows the drift uses the next step word
      ctl[TD_CTL_LAGOK] = 1u;   // ... and may use the membrane totals of the evaluation before it (PAPER.md:156 variant)
    }
    float4 p = st.pos[i];
    if (mode != 0) {
      float4 v = st.vel[i];
      float4 l = st.lo[i];
      uint32_t meta = __float_as_uint(l.w);
      float cxv[S > 1 ? S - 1 : 1];
#pragma unroll
      for (int s = 1; s < S; ++s) cxv[s - 1] = st.cx[(int64_t)(s - 1) * n + i];
      if (mode >= 2) td_half_kick<S>(P, p, v, cxv, F4, Qx, Fb, meta, i, n);
      if (mode <= 2) {
        td_half_kick<S>(P, p, v, cxv, F4, Qx, Fb, meta, i, n);
        td_drift(p.x, l.x, P.dt, v.x, P.box[0]);
        td_drift(p.y, l.y, P.dt, v.y, P.box[1]);
        td_drift(p.z, l.z, P.dt, v.z, P.box[2]);
        st.pos[i] = p;
        st.lo[i] = l;
      }
      st.vel[i] = v;
#pragma unroll
      for (int s = 1; s < S; ++s) st.cx[(int64_t)(s - 1) * n + i] = cxv[s - 1];
      if (LISTM && mode <= 2) {
        // records of the pair kernel in the slots of the last binning: exact in fp64, rounded once (as k_reorder's)
        const uint32_t pc = __ldg(&LR.rank_cell[__ldg(&LR.okey[i])]);
        const double o[3] = {(double)((float)(pc & 1022u) * P.edge_q[0]), (double)((float)((pc >> 10) & 1022u) * P.edge_q[1]),
                             (double)((float)((pc >> 20) & 1022u) * P.edge_q[2])};
        const double xa[3] = {(double)p.x + (double)l.x, (double)p.y + (double)l.y, (double)p.z + (double)l.z};
        const float4 r0 = __ldg(&LR.P4ref[i]);
        const float ref[3] = {r0.x, r0.y, r0.z};
        float rel[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          // the periodic image next to where the particle was at the binning (it moved by less than the skin)
          double t = xa[a] - o[a];
          const double L = (double)P.box[a];
          t -= L * rint((t - (double)ref[a]) / L);
          rel[a] = (float)t;
        }
        const float4 pr = make_float4(rel[0], rel[1], rel[2], p.w);
        const float4 xr = make_float4(v.w, S > 1 ? cxv[0] : 0.0f, __uint_as_float(meta & 3u), __uint_as_float(meta >> 2));
        LR.rec.P4[i] = pr;
        LR.rec.R8[2 * i] = pr;
        LR.rec.R8[2 * i + 1] = xr;
#pragma unroll
        for (int g = 0; g < td_species_groups(S); ++g) {
          float y[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) y[k] = (2 + 4 * g + k < S) ? cxv[(2 + 4 * g + k < S) ? 1 + 4 * g + k : 0] : 0.0f;
          LR.rec.Y4[(size_t)g * n + i] = make_float4(y[0], y[1], y[2], y[3]);
        }
        const float ex = rel[0] - r0.x, ey = rel[1] - r0.y, ez = rel[2] - r0.z;
        d2 = fmaf(ez, ez, fmaf(ey, ey, ex * ex));
      }
    }
    if (mode <= 2) {
      keys[i] = td_key_of(P, p.x, p.y, p.z, cell_rank);
      vals[i] = (uint32_t)i;
    }
  }
  if (LISTM && mode != 0 && mode <= 2) {  // maximum displacement: warp max, one integer atomicMax per warp (order-free)
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, d));
    if ((threadIdx.x & 31) == 0 && d2 > 0.0f) atomicMax(&ctl[TD_CTL_DMAX2], __float_as_uint(d2));
  }
}

static void launch_integrate(const DevParams& P, const SortedState& s, const float4* F4, const float* Qx,
                             const float4* Fb, int64_t n, uint32_t* keys, uint32_t* vals, const uint32_t* cell_rank,
                             int mode, uint32_t* ctl, const ListRefresh* LR, cudaStream_t st) {
  if (n == 0) return;
  int nb = (int)((n + 255) / 256);
  if (LR) {
    TD_SWITCH_S(P.n_species, k_integrate<S_, true><<<nb, 256, 0, st>>>(P, s, F4, Qx, Fb, n, keys, vals, cell_rank, mode, ctl, *LR));
  } else {
    ListRefresh none = {};
    TD_SWITCH_S(P.n_species, k_integrate<S_, false><<<nb, 256, 0, st>>>(P, s, F4, Qx, Fb, n, keys, vals, cell_rank, mode, ctl, none));
  }
}

void td_launch_init_keys(const DevParams& P, const SortedState& s, int64_t n, uint32_t* keys, uint32_t* vals,
                         const uint32_t* cell_rank, cudaStream_t st) {
  launch_integrate(P, s, nullptr, nullptr, nullptr, n, keys, vals, cell_rank, 0, nullptr, nullptr, st);
}
void td_launch_kick_drift_key(const DevParams& P, const SortedState& s, const float4* F4, const float* Qx,
                              const float4* Fb, int64_t n, uint32_t* keys, uint32_t* vals, const uint32_t* cell_rank,
                              bool closing_first, uint32_t* ctl, const ListRefresh* LR, cudaStream_t st) {
  launch_integrate(P, s, F4, Qx, Fb, n, keys, vals, cell_rank, closing_first ? 2 : 1, ctl, LR, st);
}
void td_launch_kick(const DevParams& P, const SortedState& s, const float4* F4, const float* Qx, const float4* Fb,
                    int64_t n, cudaStream_t st) {
  launch_integrate(P, s, F4, Qx, Fb, n, nullptr, nullptr, nullptr, 3, nullptr, nullptr, st);
}
