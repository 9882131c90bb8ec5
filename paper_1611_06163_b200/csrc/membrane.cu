// membrane.cu — rows a5-a8 of SURVEY §8(a): the RBC membrane bonded forces.
//   a5  bonds: WLC (Eq 13) + POW (Eq 14) springs, dissipative (Eq 15) and random (Eq 16, R10) bond forces
//   a6  K-Gather: total area / volume of each membrane, fp64, warp shuffle -> block reduce
//   a7  K-Apply: local + global area and global volume constraints (Eq 17-18) with the current step's totals (R20)
//   a8  dihedral bending (Eq 19)
// One launch.  A membrane is handled by `nchunk` CTAs; each stages all vertices of its membrane in shared memory
// (unwrapped by minimum image relative to vertex 0 and stored RELATIVE to it in fp64, exactly; every edge vector is
// the fp32 rounding of an exact difference), reduces area and volume redundantly in the same fixed order,
// and then every thread owns one vertex and recomputes the elements incident to it ("computed 3
// times, once per vertex thread" — no inter-thread communication, no atomics, fixed summation order).
#include "common.cuh"

namespace {

struct V3 { float x, y, z; };
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V3 cross3(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
__device__ __forceinline__ float dot3(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
// vertex positions are staged in fp64: a difference of two staged vertices is then exact and is rounded ONCE to fp32
// (relative error 6e-8 of the edge); positions rounded to fp32 relative to vertex 0 carry 2.4e-7 ABSOLUTE, which the
// bending term (k_b / triangle height ~ 200) turns into 3e-3 in the force
struct D3 { double x, y, z; };
__device__ __forceinline__ V3 edge(const D3& a, const D3& b) { return {(float)(a.x - b.x), (float)(a.y - b.y), (float)(a.z - b.z)}; }
__device__ __forceinline__ V3 tof(const D3& a) { return {(float)a.x, (float)a.y, (float)a.z}; }

// minimum-image difference a - b of two wrapped fp32 coordinates, exact in fp64
__device__ __forceinline__ double min_image_diff(float a, float b, float L) {
  double d = (double)a - (double)b;
  if (d > 0.5 * (double)L) d -= (double)L;
  else if (d < -0.5 * (double)L) d += (double)L;
  return d;
}

// dU_WLC/dh = (kBT/p) (1/(4(1-x)^2) - 1/4 + x)   (from Eq 13)
__device__ __forceinline__ float wlc_force(float kBT_over_p, float x) {
  float om = 1.0f - x;
  return kBT_over_p * (0.25f / (om * om) - 0.25f + x);
}

// 64 registers (four CTAs per SM) instead of the 128 ptxas takes when left alone (two CTAs, 19 % occupancy): the kernel
// is bound by fixed-latency and load waits at IPC 1.8, not by registers; config 5: 0.258 -> 0.208 ms alone, the step
// 6.478 -> 6.433 ms with the kernel beside the pair kernel (3 and 5 CTAs per SM: 6.447 / 6.439)
#ifndef TD_MEM_MINB
#define TD_MEM_MINB 4
#endif
__global__ void __launch_bounds__(256, TD_MEM_MINB) k_membrane(const __grid_constant__ DevParams P, const MembraneArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[2][8];
  __shared__ double tot[2];
  const uint32_t step = __ldg(A.step_p);
  const int m = blockIdx.x / A.nchunk, chunk = blockIdx.x % A.nchunk;
  const RbcDev R = A.rbcs[m];
  const MeshTemplateDev T = A.tmpls[R.tmpl];
  const int nv = T.nv, t = threadIdx.x, NT = blockDim.x, lane = t & 31, warp = t >> 5;
  D3* sr = (D3*)smem_raw;                         // [nv] unwrapped positions relative to vertex 0 (fp64, exact)
  V3* sv = (V3*)(smem_raw + (size_t)nv * 24);     // [nv] velocities

  // ---- stage vertices (gather through slot_of_id)
  const uint32_t slot0 = A.slot_of_id[R.first_id];
  const float4 p0 = A.st.pos[slot0];
  const float4 l0 = A.st.lo[slot0];
  for (int v = t; v < nv; v += NT) {
    uint32_t slot = A.slot_of_id[R.first_id + v];
    float4 p = A.st.pos[slot];
    float4 l = A.st.lo[slot];
    float4 w = A.st.vel[slot];
    sr[v] = {min_image_diff(p.x, p0.x, P.box[0]) + ((double)l.x - (double)l0.x),
             min_image_diff(p.y, p0.y, P.box[1]) + ((double)l.y - (double)l0.y),
             min_image_diff(p.z, p0.z, P.box[2]) + ((double)l.z - (double)l0.z)};
    sv[v] = {w.x, w.y, w.z};
  }
  __syncthreads();

  // ---- a6 K-Gather in fp64 (fixed order: thread-strided partials, shuffle tree, warps in order)
  double aA = 0.0, aV = 0.0;
  for (int k = t; k < T.ntri; k += NT) {
    D3 a = sr[T.tri[3 * k]], b = sr[T.tri[3 * k + 1]], c = sr[T.tri[3 * k + 2]];
    double ax = a.x, ay = a.y, az = a.z, bx = b.x, by = b.y, bz = b.z, cx = c.x, cy = c.y, cz = c.z;
    double ux = bx - ax, uy = by - ay, uz = bz - az, wx = cx - ax, wy = cy - ay, wz = cz - az;
    double nx = uy * wz - uz * wy, ny = uz * wx - ux * wz, nz = ux * wy - uy * wx;
    aA += 0.5 * sqrt(nx * nx + ny * ny + nz * nz);
    aV += (ax * (by * cz - bz * cy) + ay * (bz * cx - bx * cz) + az * (bx * cy - by * cx)) * (1.0 / 6.0);
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    aA += __shfl_down_sync(0xffffffffu, aA, d);
    aV += __shfl_down_sync(0xffffffffu, aV, d);
  }
  if (lane == 0) { red[0][warp] = aA; red[1][warp] = aV; }
  __syncthreads();
  if (t == 0) {
    double sA = 0.0, sV = 0.0;
    for (int w = 0; w < (NT + 31) / 32; ++w) { sA += red[0][w]; sV += red[1][w]; }
    const int M = gridDim.x / A.nchunk;
    double* cur = A.stats + (size_t)(step & 1u) * 2 * M;
    if (chunk == 0) { cur[2 * m] = sA; cur[2 * m + 1] = sV; }
    // K-Apply totals: this evaluation's (sequential variant, R20) or, those of the previous step's
    // evaluation (written by an earlier launch, so that K-Apply does not depend on this launch's reduction)
    if (A.lag_av && A.step_p[TD_CTL_LAGOK]) {
      const double* lag = A.stats + (size_t)((step & 1u) ^ 1u) * 2 * M;
      sA = lag[2 * m]; sV = lag[2 * m + 1];
    }
    tot[0] = sA; tot[1] = sV;
  }
  __syncthreads();
  const float beta_g = (float)(-(double)R.k_g * (tot[0] - R.A0) / R.A0);
  const float beta_v6 = (float)(-(double)R.k_v * (tot[1] - R.V0) / R.V0 / 6.0);

  // ---- per-vertex forces
  const int CH = (nv + A.nchunk - 1) / A.nchunk;
  const int vend = min(nv, (chunk + 1) * CH);
  const float* h0 = A.h0 + R.data_off;
  const float* kp = A.kp + R.data_off;
  const float* A0t = A.A0t + R.tri_off;
  for (int v = chunk * CH + t; v < vend; v += NT) {
    const D3 rv = sr[v];
    const V3 vv = sv[v];
    float fx = 0.f, fy = 0.f, fz = 0.f;
    const int e0 = T.voff[v], e1 = T.voff[v + 1];
    // a5 bonds (Eq 13-16): force on v from bond (v,u), d = r_v - r_u
    for (int e = e0; e < e1; ++e) {
      uint32_t pk = T.vbond[e];
      int u = pk & 0xFFFFu, b = pk >> 16;
      V3 d = edge(rv, sr[u]), dv = vv - sv[u];
      float h2 = dot3(d, d), hinv = rsqrtf(h2), h = h2 * hinv;
      V3 ev = {d.x * hinv, d.y * hinv, d.z * hinv};
      float x = h * R.inv_x0 / h0[b];
      if (x >= 1.0f) atomicOr(A.err, TD_ERR_BOND_OVERSTRETCH);
      float fpow = R.m_pow == 2.0f ? kp[b] * hinv * hinv : kp[b] * exp2f(-R.m_pow * __log2f(h));
      float f = -wlc_force(R.kBT_over_p, x) + fpow;
      float edv = dot3(ev, dv);
      // random part: N rows from Philox tags 1,2,3 of (min id, max id, step)
      uint32_t ia = (uint32_t)(R.first_id + v), ib = (uint32_t)(R.first_id + u);
      uint32_t lo = min(ia, ib), hi = max(ia, ib);
      float N[9];
#pragma unroll
      for (int row = 0; row < 3; ++row) {
        uint32_t x0, x1, x2, x3;
        float g0, g1, g2, g3;
        td_philox(lo, hi, step, 1u + row, P.key0, P.key1, x0, x1, x2, x3);
        td_box_muller(x0, x1, g0, g1);
        td_box_muller(x2, x3, g2, g3);
        N[3 * row] = g0; N[3 * row + 1] = g1; N[3 * row + 2] = g2;
      }
      float tr = N[0] + N[4] + N[8];
      float diag = R.rnd_C * tr - R.rnd_T * tr * (1.0f / 3.0f);
      float s01 = 0.5f * (N[1] + N[3]), s02 = 0.5f * (N[2] + N[6]), s12 = 0.5f * (N[5] + N[7]);
      float rx = R.rnd_T * (N[0] * ev.x + s01 * ev.y + s02 * ev.z) + diag * ev.x;
      float ry = R.rnd_T * (s01 * ev.x + N[4] * ev.y + s12 * ev.z) + diag * ev.y;
      float rz = R.rnd_T * (s02 * ev.x + s12 * ev.y + N[8] * ev.z) + diag * ev.z;
      float fe = f - R.gamma_C * edv;
      fx += fe * ev.x - R.gamma_T * dv.x + rx;
      fy += fe * ev.y - R.gamma_T * dv.y + ry;
      fz += fe * ev.z - R.gamma_T * dv.z + rz;
    }
    // a7 K-Apply (Eq 17-18): triangles incident to v; role k: p_k = v, pa = p_{k+1}, pb = p_{k+2}
    for (int e = e0; e < e1; ++e) {
      uint32_t pk = T.vtri[e];
      int tri = pk & 0xFFFFu, role = pk >> 16;
      int i1 = T.tri[3 * tri + (role + 1) % 3], i2 = T.tri[3 * tri + (role + 2) % 3];
      const D3 pad = sr[i1], pbd = sr[i2];
      V3 pa = tof(pad), pb = tof(pbd);
      V3 xi = cross3(edge(pad, rv), edge(pbd, rv));  // same normal for any cyclic start
      float l2 = dot3(xi, xi), linv = rsqrtf(l2);
      float At = 0.5f * l2 * linv;
      float a0 = A0t[tri];
      float beta = beta_g - R.k_l * (At - a0) / a0;
      V3 nh = {xi.x * linv, xi.y * linv, xi.z * linv};
      V3 ga = cross3(nh, edge(pbd, pad)), gv = cross3(pa, pb);
      fx += 0.5f * beta * ga.x + beta_v6 * gv.x;
      fy += 0.5f * beta * ga.y + beta_v6 * gv.y;
      fz += 0.5f * beta * ga.z + beta_v6 * gv.z;
    }
    // a8 bending (Eq 19): dihedrals in which v takes part
    for (int e = T.vdoff[v]; e < T.vdoff[v + 1]; ++e) {
      uint32_t pk = T.vdih[e];
      int q = pk & 0xFFFFu, role = pk >> 16;
      D3 r1 = sr[T.dih[4 * q]], r2 = sr[T.dih[4 * q + 1]], r3 = sr[T.dih[4 * q + 2]], r4 = sr[T.dih[4 * q + 3]];
      // the two triangle normals in fp64 from the exact edge differences
      V3 ee = edge(r3, r2);
      double ax = r2.x - r1.x, ay = r2.y - r1.y, az = r2.z - r1.z;
      double bx = r3.x - r1.x, by = r3.y - r1.y, bz = r3.z - r1.z;
      double cx = r3.x - r4.x, cy = r3.y - r4.y, cz = r3.z - r4.z;
      double dx = r2.x - r4.x, dy = r2.y - r4.y, dz = r2.z - r4.z;
      double xid[3] = {ay * bz - az * by, az * bx - ax * bz, ax * by - ay * bx};
      double zed[3] = {cy * dz - cz * dy, cz * dx - cx * dz, cx * dy - cy * dx};
      double xi2d = xid[0] * xid[0] + xid[1] * xid[1] + xid[2] * xid[2];
      double ze2d = zed[0] * zed[0] + zed[1] * zed[1] + zed[2] * zed[2];
      double cd = xid[0] * zed[0] + xid[1] * zed[1] + xid[2] * zed[2];
      double sd = (xid[1] * zed[2] - xid[2] * zed[1]) * ee.x + (xid[2] * zed[0] - xid[0] * zed[2]) * ee.y +
                  (xid[0] * zed[1] - xid[1] * zed[0]) * ee.z;
      V3 xi = {(float)xid[0], (float)xid[1], (float)xid[2]}, ze = {(float)zed[0], (float)zed[1], (float)zed[2]};
      float xi2 = (float)xi2d, ze2 = (float)ze2d, e2 = dot3(ee, ee);
      float le = sqrtf(e2);
      double ixzd = rsqrt(xi2d * ze2d);
      float cth = (float)(cd * ixzd);
      float sth = (float)(sd * ixzd) / le;
      // sin(theta - theta0) with (cos, sin) normalised (they are, up to rounding)
      float nrm = rsqrtf(cth * cth + sth * sth);
      float coef = -R.k_b * (sth * R.cos_t0 - cth * R.sin_t0) * nrm;
      float c1 = -le / xi2, c4 = -le / ze2;  // g1 = c1 xi, g4 = c4 ze
      float w1, w4;
      if (role == 0) { w1 = 1.f; w4 = 0.f; }
      else if (role == 3) { w1 = 0.f; w4 = 1.f; }
      else {
        float s1 = dot3(edge(r1, r2), ee) / e2, s4 = dot3(edge(r4, r2), ee) / e2;
        if (role == 1) { w1 = -(1.f - s1); w4 = -(1.f - s4); }
        else { w1 = -s1; w4 = -s4; }
      }
      float k1 = coef * w1 * c1, k4 = coef * w4 * c4;
      fx += k1 * xi.x + k4 * ze.x;
      fy += k1 * xi.y + k4 * ze.y;
      fz += k1 * xi.z + k4 * ze.z;
    }
    A.Fb[R.first_id + v] = make_float4(fx, fy, fz, 0.f);
  }
}
}  // namespace

int td_launch_membrane(const DevParams& P, const MembraneArgs& A, int n_rbc, int max_nv, int nthreads,
                       cudaStream_t st) {
  if (n_rbc == 0) return 0;
  size_t smem = (size_t)max_nv * 36;
  cudaError_t e = cudaFuncSetAttribute(k_membrane, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return (int)e;
  k_membrane<<<n_rbc * A.nchunk, nthreads, smem, st>>>(P, A);
  return 0;
}
