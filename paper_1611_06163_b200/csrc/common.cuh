// common.cuh — device-side structures shared by the kernels of libtdpd.so (CUDA path only; nothing here is
// shared with oracle/).  Citations: /root/reference/PAPER.md:<line>, readings R<n>.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define TD_T 4  // max particle types
#define TD_S 10  // max species (the paper benchmarks up to N_spec = 10)

// Parameters in the form the kernels consume (derived once on the host from tdpd_params).
struct DevParams {
  int n_types, n_species;
  float box[3];
  float half_box_z;
  int ncell[3];
  float cell_inv[3];   // (float)(n_a / L_a): binning multiplier (R-bin)
  float cell_edge[3];  // L_a / n_a
  // pair-kernel coordinates are stored RELATIVE to the origin of the particle's 2x2x2 cell block,
  // o = (c & ~1) * edge_q (exact in fp32: edge_q keeps 13 significant bits and c < 1024), so that differences
  // between neighbouring blocks are exact; gap = L - n edge_q (kept for reference)
  float edge_q[3], gap[3];
  float r_c, r_cc, rc2, rcc2, rcut2, inv_rc, inv_rcc;
  float dt, half_dt;
  // type-pair tables, index ti*TD_T + tj
  float a[TD_T * TD_T];
  float gamma[TD_T * TD_T];
  float sig[TD_T * TD_T];  // sqrt(2 kBT gamma) / sqrt(dt)   (Eq 5-6)
  float s_R[TD_T * TD_T];
  float kappa[TD_S][TD_T * TD_T];
  float epsc[TD_S];  // m_s^2 rho / dt: Q^R = sgn zeta w_RC sqrt(kappa (Ci+Cj) epsc)  (Eq 9-10)
  float epsc2[TD_S];  // -2 ln 2 * epsc: multiplies lg2(u) so that sqrt(-2 ln u) and the amplitude share one square root
  float s_c[TD_S];
  float body[3];
  int body_mode;
  uint32_t key0[10], key1[10];  // Philox round keys: seed + r * Weyl
  int excl_same;
  int fast_w;     // every s_R == 0.5 and every s_c == 2: weights need no pow
  int rand_flux;  // some m_s != 0
  int has_source; // some source / decay rate != 0
  float src[TD_S][TD_T], dec[TD_S][TD_T];  // Q^S_i = src[s][type] - dec[s][type] C_i^s  (Eq 7, reading R-QS)
};

// meta word of a particle: bits 0-1 type, bits 2-31 membrane id + 1 (0 = free particle)
__host__ __device__ inline uint32_t td_meta(int type, int rbc1) { return (uint32_t)type | ((uint32_t)rbc1 << 2); }

// ---- Philox-4x32-10 (Salmon et al. SC'11; DESIGN.md R-RNG) -----------------------------------------------
// counter (c0,c1,c2,c3), round keys precomputed in DevParams.
__device__ __forceinline__ void td_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t* k0,
                                          const uint32_t* k1, uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0[r];
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1[r];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
  }
  o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// word -> uniform strictly inside (0,1): u = ((x >> 9) + 1/2) 2^-23 (exact in fp32)
// evaluated without an int->float conversion: 1.m - (1 - 2^-24) with m = x >> 9 is exact (Sterbenz + 24-bit result)
__device__ __forceinline__ float td_uniform(uint32_t x) {
  return __uint_as_float((x >> 9) | 0x3f800000u) - 0.99999994039535522f;
}
__device__ __forceinline__ float td_sqrt_approx(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float td_rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ float td_rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float td_lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float td_sin_approx(float x) {
  float y;
  asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float td_cos_approx(float x) {
  float y;
  asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Box-Muller: R = sqrt(-2 ln ua); (g_cos, g_sin) = R (cos 2 pi ub, sin 2 pi ub).
// MUFU lg2/sqrt/sin/cos; lg2.approx has absolute error 2^-22 on (0.5, 2), which is not good enough for R when
// ua -> 1 (R -> 0), so the top 2^-10 of the range uses the series of -2 ln(1 - t) with t = 1 - ua (exact in fp32).
// Branch-free.
// radius from the uniform u and its lg2 (shared by the pair kernel, which needs lg2(u) for the flux as well)
__device__ __forceinline__ float td_bm_radius_l(float u, float lg2u) {
  const float t = 1.0f - u;
  const float q1 = -1.3862943611198906f * lg2u;  // -2 ln 2 * lg2(u)
  // -2 ln(1 - t) = 2 t + t^2 + 2/3 t^3 + O(t^4): below t = 2^-10 the series is exact to 3e-10 relative, while the
  // 2^-22 absolute error of lg2.approx would be 2e-4 of q at t = 2^-10 and 1 % at t = 2^-16 (measured, round 2)
  const float q2 = t * fmaf(t, fmaf(t, 0.66666669f, 1.0f), 2.0f);
  return td_sqrt_approx(t < 9.765625e-04f ? q2 : q1);
}
__device__ __forceinline__ float td_bm_radius(uint32_t xa) {
  const float u = td_uniform(xa);
  return td_bm_radius_l(u, td_lg2_approx(u));
}
__device__ __forceinline__ void td_box_muller(uint32_t xa, uint32_t xb, float& g_cos, float& g_sin) {
  const float R = td_bm_radius(xa);
  const float ang = 6.283185307179586f * td_uniform(xb);
  g_cos = R * td_cos_approx(ang);
  g_sin = R * td_sin_approx(ang);
}

// cheapest variant, without the u -> 1 series: for the random-flux Gaussians of ring entries, whose amplitude
// m_s sqrt(kappa rho C / dt) is ~1e-2 of the Fickian flux, so the 5e-5 absolute error of lg2.approx near u = 1 is nil
__device__ __forceinline__ void td_box_muller_fast(uint32_t xa, uint32_t xb, float& g_cos, float& g_sin) {
  const float R = td_sqrt_approx(-1.3862943611198906f * td_lg2_approx(td_uniform(xa)));
  const float ang = 6.283185307179586f * td_uniform(xb);
  g_cos = R * td_cos_approx(ang);
  g_sin = R * td_sin_approx(ang);
}

// ---- kernel argument blocks -----------------------------------------------------------------------------
struct SortedState {   // one side of the ping-pong, cell-sorted order
  float4* pos;     // x, y, z, id (bits)
  float4* vel;     // vx, vy, vz, C_0
  float* cx;       // [(S-1)][n]: C_1.. species-major
  float4* lo;      // low-order words of x, y, z (position = pos + lo, two-float), td_meta (bits)
};

// pair-kernel records, written by the reorder kernel in cell-sorted order (read-only in the pair kernel)
struct PairRec {
  float4* P4;   // x, y, z relative to the origin of the 2x2x2 cell block, (c & ~1) * edge_q (see DevParams), id (bits)
  float4* R8;   // [2n] the record the evaluation loads with ONE 256-bit load (LDG.E.256, new on sm_100) per neighbour:
                // R8[2i] = P4[i], R8[2i+1] = C_0, C_1, type (bits), exclusion key = membrane id + 1 or 0 (bits)
  float4* Y4;   // [td_species_groups(S)][n]: C_2..C_5, C_6..C_9 (species-major in groups of four; zero padded)
};

// the pair kernel is compiled for 1, 2, 4, 6 and 10 species; other counts run the next larger one (a padded species has
// kappa = 0 and C = 0: its flux is exactly zero and is never stored)
__host__ __device__ constexpr int td_species_padded(int S) { return S <= 2 ? S : S <= 4 ? 4 : S <= 6 ? 6 : 10; }
__host__ __device__ constexpr int td_species_groups(int S) { return S <= 2 ? 0 : (td_species_padded(S) - 2 + 3) / 4; }

// device control words (one 64-word block; word 0 is the RNG step word the integrator bumps)
enum { TD_CTL_STEP = 0, TD_CTL_REBUILD = 1, TD_CTL_DMAX2 = 2, TD_CTL_FORCE = 3, TD_CTL_NREBUILD = 4, TD_CTL_NDECIDE = 5,
       TD_CTL_LAGOK = 6 };  // LAGOK: the membrane totals of the previous step's force evaluation exist

// what the integrator needs to keep the pair records current between binnings (neighbour-list mode)
struct ListRefresh {
  const uint32_t* okey;       // [n] Morton rank of the cell each slot was binned into
  const uint32_t* rank_cell;  // [ncell]
  PairRec rec;
  const float4* P4ref;        // [n] P4 at the last binning (displacement reference)
};

struct PairArgs {
  PairRec rec;
  const float4* vel;           // vx, vy, vz, C_0 (SortedState::vel)
  const float4* pos;           // hi words of the positions (SortedState::pos)
  const float4* lo;            // low words (SortedState::lo)
  const uint32_t* keys;        // [n] Morton rank of the cell of each slot (sorted)
  const uint32_t* cell_start;  // [ncell + 1] by Morton rank
  const uint32_t* cell_rank;   // [ncell] x-fastest linear cell -> Morton rank
 const uint32_t* rank_cell;   // [ncell] Morton rank -> packed cx | cy << 10 | cz << 20
  // static neighbour segments of every cell (CSR by Morton rank): runs of rank-consecutive neighbour cells that
  // lie in one 2x2x2 block and one periodic image, so that one displacement serves the whole run
  const uint32_t* seg_off;     // [ncell + 1]
  const uint32_t* seg_first;   // first Morton rank of the run
  const uint32_t* seg_meta;    // cells in the run | (wrap_x + 1) << 4 | (wrap_y + 1) << 6 | (wrap_z + 1) << 8
  float4* F4;                  // Fx, Fy, Fz, Q_0 by slot
  float* Qx;                   // [(S-1)][n]
  int64_t n;
  const uint32_t* step_p;      // RNG step word (device counter, bumped by the integrator: lets a step be a CUDA graph)
  int lcap;                    // list entries per thread
  int* err;                    // device error word
  // neighbour list reused between binnings: tiles of 256 slots, [tile][entry][lane], 16-bit
  // entries run << 11 | offset against the cell table of the binning that built it
  uint16_t* nlist;
  uint32_t* nl_cnt;            // [n] entries of each slot
  int nl_cap;                  // entries per slot
  float rlist2;                // (max(r_c, r_cc) + skin)^2
  uint32_t* census;            // test support: [4][n] by id (front count, front id xor, ring count, ring id xor) or NULL
};

// mesh template (topology shared by all membranes with the same triangle list), CSR per vertex
struct MeshTemplateDev {
  int nv, ntri, nbond;
  const uint16_t* tri;    // [ntri][3]
  const uint16_t* dih;    // [nbond][4]
  const int* voff;        // [nv + 1]
  const uint32_t* vbond;  // [2 nbond]: neighbour vertex | bond index << 16
  const uint32_t* vtri;   // [3 ntri]: triangle | role << 16
  const int* vdoff;       // [nv + 1]
  const uint32_t* vdih;   // [4 nbond]: dihedral | role << 16
};

struct RbcDev {
  int64_t first_id;
  int tmpl;
  int data_off;  // offset of this membrane's h0/kp (per bond) arrays
  int tri_off;   // offset of A0t
  double A0, V0;  // fp64: (A - A0) / A0 is multiplied by k_g ~ 2e4, an fp32 A0 alone would cost 1e-3 in beta
  float kBT_over_p, inv_x0, m_pow, gamma_T, gamma_C, k_g, k_l, k_v, k_b, cos_t0, sin_t0;
  float rnd_T, rnd_C;  // sqrt(2 kBT/dt) sqrt(2 gT), sqrt(2 kBT/dt) sqrt(3 gC - gT)/3
};

struct MembraneArgs {
  SortedState st;
  const uint32_t* slot_of_id;
  const RbcDev* rbcs;
  const MeshTemplateDev* tmpls;
  const float* h0;
  const float* kp;
  const float* A0t;
  float4* Fb;       // bonded force by id
  double* stats;    // [2][M][2] area, volume of the force evaluation with step word k in slot k & 1
  int lag_av;       // PAPER.md:156 variant: K-Apply with the totals of the previous step's evaluation (slot (k - 1) & 1)
  int nchunk;       // CTAs per membrane
  const uint32_t* step_p;  // RNG step word (device counter)
  int* err;
};

enum { TD_ERR_CELL_OVERFLOW = 1, TD_ERR_NONFINITE = 2, TD_ERR_BOND_OVERSTRETCH = 4, TD_ERR_LIST_OVERFLOW = 8 };

#ifndef TD_PAIR_MAXLOC
#define TD_PAIR_MAXLOC 24  // cells per neighbour-table chunk of the pair kernel (a 256-slot blob spans ~20)
#endif
// shared memory of the pair kernel ahead of the hit stacks: run table (first slot + displacement 16 B, count 4 B per
// run), type-pair table (a, gamma, sigma, s_R), kappa per species, runs per local cell
__host__ __device__ constexpr size_t td_pair_table_bytes() {
  return (size_t)TD_PAIR_MAXLOC * 27 * 20 + 16 * 16 + (size_t)TD_S * 16 * 4 + TD_PAIR_MAXLOC * 4;
}

// runs `...` with the compile-time species count S_ = ns (1..TD_S)
#define TD_SWITCH_S(ns, ...)                                       \
  switch (ns) {                                                    \
    case 1: { constexpr int S_ = 1; __VA_ARGS__; } break;          \
    case 2: { constexpr int S_ = 2; __VA_ARGS__; } break;          \
    case 3: { constexpr int S_ = 3; __VA_ARGS__; } break;          \
    case 4: { constexpr int S_ = 4; __VA_ARGS__; } break;          \
    case 5: { constexpr int S_ = 5; __VA_ARGS__; } break;          \
    case 6: { constexpr int S_ = 6; __VA_ARGS__; } break;          \
    case 7: { constexpr int S_ = 7; __VA_ARGS__; } break;          \
    case 8: { constexpr int S_ = 8; __VA_ARGS__; } break;          \
    case 9: { constexpr int S_ = 9; __VA_ARGS__; } break;          \
    default: { constexpr int S_ = 10; __VA_ARGS__; } break;        \
  }

// ---- launchers (each .cu exposes host functions; all launches are asynchronous on `st`) -------------------
void td_launch_init_keys(const DevParams& P, const SortedState& s, int64_t n, uint32_t* keys, uint32_t* vals,
                         const uint32_t* cell_rank, cudaStream_t st);
void td_launch_kick_drift_key(const DevParams& P, const SortedState& s, const float4* F4, const float* Qx,
                              const float4* Fb, int64_t n, uint32_t* keys, uint32_t* vals, const uint32_t* cell_rank,
                              bool closing_first, uint32_t* ctl, const ListRefresh* LR, cudaStream_t st);
void td_launch_kick(const DevParams& P, const SortedState& s, const float4* F4, const float* Qx, const float4* Fb,
                    int64_t n, cudaStream_t st);
int td_sort_passes(int key_bits);
size_t td_sort_scratch_bytes(int64_t n);
// sorts (keys, vals); result ends in keys[out_side]/vals[out_side]; returns out_side
int td_launch_sort(uint32_t* keys[2], uint32_t* vals[2], int64_t n, int key_bits, void* scratch, cudaStream_t st,
                   int* n_launches, const uint32_t* gate);
void td_launch_reorder(const DevParams& P, const SortedState& src, const SortedState& dst, const PairRec& rec,
                       const uint32_t* keys, const uint32_t* vals, const uint32_t* rank_cell, int64_t n,
                       uint32_t ncell, uint32_t* cell_start, uint32_t* slot_of_id, uint32_t* okey, float4* P4ref,
                       const uint32_t* gate, cudaStream_t st);
void td_launch_copy_state(const DevParams& P, const SortedState& src, const SortedState& dst, int64_t n,
                          const uint32_t* gate, cudaStream_t st);
// neighbour-list mode (pair_list.cu): the per-step decision and the list builder
void td_launch_list_decide(uint32_t* ctl, float skin2, cudaStream_t st);
int td_launch_build_list(const DevParams& P, const PairArgs& A, const uint32_t* gate, cudaStream_t st);
int td_launch_pair(const DevParams& P, const PairArgs& A, int nthreads, int split, bool from_list, cudaStream_t st);
size_t td_pair_smem_bytes(int lcap, int nthreads);
int td_launch_membrane(const DevParams& P, const MembraneArgs& A, int n_rbc, int max_nv, int nthreads,
                       cudaStream_t st);
void td_launch_unsort(const SortedState& s, const float4* F4, const float* Qx, const float4* Fb, int64_t n,
                      int n_species, int what, float* out, int* err, const float* box, cudaStream_t st);
void td_launch_set_state(const DevParams& P, const SortedState& s, int64_t n, const float* pos, const float* vel,
                         const float* conc, cudaStream_t st);
void td_launch_binning_debug(const DevParams& P, const SortedState& s, int64_t n, const uint32_t* keys,
                             const uint32_t* rank_cell, int32_t* cell_xyz, int32_t* cell_count, int32_t* sorted_id,
                             cudaStream_t st);
void td_launch_census(const DevParams& P, const SortedState& s, const uint32_t* cell_start, const uint32_t* cell_rank,
                      const uint32_t* keys, const uint32_t* rank_cell, int64_t n, int32_t* n_rc, int32_t* n_rcc,
                      uint32_t* xor_rc, uint32_t* xor_rcc, cudaStream_t st);
void td_launch_rng_debug(const DevParams& P, int64_t n, const int64_t* id_i, const int64_t* id_j, uint32_t step,
                         uint32_t tag, uint32_t* words, float* gauss, cudaStream_t st);
void td_launch_box_muller_debug(int64_t n, const uint32_t* words, float* gauss, cudaStream_t st);
