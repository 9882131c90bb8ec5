// api.cu — host side of libtdpd.so: the C ABI of include/tdpd.h, workspace layout, derived membrane topology and
// the step orchestration (two streams joined by events).  No arithmetic of the method runs
// on the host after upload; the host only derives constants and index tables.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "../../include/tdpd.h"
#include "common.cuh"

namespace {

struct MeshTemplate {
  int nv = 0, ntri = 0, nbond = 0;
  std::vector<int32_t> tri;        // [ntri][3] as given
  std::vector<int32_t> bond, dih;  // [nbond][2], [nbond][4]
  std::vector<uint16_t> tri16, dih16;
  std::vector<int> voff, vdoff;
  std::vector<uint32_t> vbond, vtri, vdih;
};

struct RbcHost {
  int64_t first_id;
  int tmpl, nv;
  tdpd_rbc_params rp;
  std::vector<float> h0, kp, A0t;
  double A0, V0;
};

struct Timer {
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev;
  int64_t launches = 0;
  double ms = 0.0;
};

}  // namespace

struct tdpd_sim {
  tdpd_params prm;
  DevParams dp;
  int device = 0;
  cudaStream_t sA = nullptr, sB = nullptr;
  bool own_streams = false;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  // host staging until the workspace is set
  std::vector<float> h_pos, h_vel, h_conc;
  std::vector<int32_t> h_type, h_rbc;
  std::vector<MeshTemplate> tmpls;
  std::vector<RbcHost> rbcs;
  // grid
  uint32_t ncells = 0;
  int key_bits = 0;
  std::vector<uint32_t> cell_rank, rank_cell;
  std::vector<uint32_t> seg_off, seg_first, seg_meta;  // static neighbour runs of every cell (PairArgs)
  int pair_nt = 256, lcap = 72, pair_split = 1, tune_nt = 0, tune_lcap = 0, tune_split = 0;
  PairRec rec = {nullptr, nullptr, nullptr};
  uint32_t* keys_sorted = nullptr;
  int mem_nchunk = 1, mem_nt = 256, max_nv = 0;
  bool lag_av = false;  // PAPER.md:156 variant of K-Apply
  // device
  void* ws = nullptr;
  size_t ws_bytes = 0;
  bool own_ws = false, finalized = false;
  SortedState st[2];
  int cur = 0;
  uint32_t *keys[2] = {nullptr, nullptr}, *vals[2] = {nullptr, nullptr};
  void* sort_scratch = nullptr;
  uint32_t *cell_start = nullptr, *cell_rank_d = nullptr, *rank_cell_d = nullptr, *slot_of_id = nullptr;
  uint32_t *seg_off_d = nullptr, *seg_first_d = nullptr, *seg_meta_d = nullptr;
  float4 *F4 = nullptr, *Fb = nullptr;
  float *Qx = nullptr, *staging = nullptr;
  int* err_d = nullptr;
  uint32_t* step_d = nullptr;  // device control block; word 0 = the step word (the integrator bumps it), see TD_CTL_*
  // neighbour list reused between binnings; nl_skin > 0 switches the mode on
  float nl_skin = 0.0f;
  int nl_cap = 0, tune_nl_cap = 0;
  uint16_t* nlist_d = nullptr;
  uint32_t *nl_cnt_d = nullptr, *okey_d = nullptr;
  float4* P4ref_d = nullptr;
  double* stats_d = nullptr;
  RbcDev* rbcs_d = nullptr;
  MeshTemplateDev* tmpls_d = nullptr;
  float *h0_d = nullptr, *kp_d = nullptr, *A0t_d = nullptr;
  unsigned char* topo_d = nullptr;
  int64_t n = 0, step = 0;
  bool have_forces = false, binned = false;
  bool timing = false;
  // CUDA graphs of one step, by [side of the ping-pong][first step of a call][last step of a call]
  bool use_graph = true;
  cudaGraphExec_t gexec[2][2][2] = {};
  int glaunches[2][2][2] = {};
  uint32_t* gkeys[2][2][2] = {};
  Timer timers[TDPD_N_TIMERS];
  int64_t launches = 0;
  std::string err;
};

namespace {

int fail(tdpd_sim* s, int code, const std::string& msg) {
  if (s) s->err = msg;
  return code;
}
#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(s, TDPD_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

bool validate_params(const tdpd_params* p, std::string& why) {
  if (!p || p->struct_size != sizeof(tdpd_params)) { why = "struct_size mismatch"; return false; }
  if (p->n_types < 1 || p->n_types > TDPD_MAX_TYPES || p->n_species < 1 || p->n_species > TDPD_MAX_SPECIES) {
    why = "n_types / n_species out of range"; return false;
  }
  if (!(p->r_c > 0) || !(p->r_cc > 0) || !(p->dt > 0) || !(p->kBT >= 0) || !(p->rho >= 0)) { why = "non-positive scalar"; return false; }
  double rcut = std::max(p->r_c, p->r_cc);
  for (int a = 0; a < 3; ++a) {
    int nc = (int)std::floor((double)p->box[a] / rcut);
    if (nc < 3) { why = "box smaller than 3 cells per axis"; return false; }
    if (nc > 1023) { why = "more than 1023 cells per axis"; return false; }
  }
  for (int i = 0; i < p->n_types; ++i)
    for (int j = 0; j < p->n_types; ++j) {
      if (p->a[i][j] != p->a[j][i] || p->gamma[i][j] != p->gamma[j][i] || p->s_R[i][j] != p->s_R[j][i]) { why = "asymmetric type table"; return false; }
      if (p->gamma[i][j] < 0 || p->s_R[i][j] < 0) { why = "negative gamma / s_R"; return false; }
      for (int sp = 0; sp < p->n_species; ++sp) {
        if (p->kappa[sp][i][j] != p->kappa[sp][j][i] || p->kappa[sp][i][j] < 0) { why = "asymmetric or negative kappa"; return false; }
      }
    }
  for (int sp = 0; sp < p->n_species; ++sp)
    if (p->m_s[sp] < 0 || p->s_c[sp] < 0) { why = "negative m_s / s_c"; return false; }
  if (p->body_mode < 0 || p->body_mode > 2) { why = "body_mode"; return false; }
  return true;
}

// skin > 0 (neighbour-list mode): the cells must hold every pair within cutoff + skin in the 27-cell stencil
void derive_params(const tdpd_params& p, DevParams& d, float skin = 0.0f) {
  memset(&d, 0, sizeof d);
  d.n_types = p.n_types; d.n_species = p.n_species;
  double rcut = (double)std::max(p.r_c, p.r_cc) + (double)skin;
  for (int a = 0; a < 3; ++a) {
    d.box[a] = p.box[a];
    d.ncell[a] = (int)std::floor((double)p.box[a] / rcut);
    d.cell_inv[a] = (float)((double)d.ncell[a] / (double)p.box[a]);
    d.cell_edge[a] = (float)((double)p.box[a] / (double)d.ncell[a]);
    {  // edge_q: the cell edge truncated to 13 significant bits, so that c * edge_q is exact in fp32 for c < 1024
      int ex;
      double mant = std::frexp((double)p.box[a] / (double)d.ncell[a], &ex);
      double eq = std::ldexp(std::floor(mant * 8192.0) / 8192.0, ex);
      d.edge_q[a] = (float)eq;
      d.gap[a] = (float)((double)p.box[a] - (double)d.ncell[a] * eq);
    }
    d.body[a] = p.body_force[a];
  }
  d.half_box_z = 0.5f * p.box[2];
  d.r_c = p.r_c; d.r_cc = p.r_cc;
  d.rc2 = p.r_c * p.r_c; d.rcc2 = p.r_cc * p.r_cc;
  d.rcut2 = std::max(d.rc2, d.rcc2);
  d.inv_rc = (float)(1.0 / (double)p.r_c); d.inv_rcc = (float)(1.0 / (double)p.r_cc);
  d.dt = p.dt; d.half_dt = 0.5f * p.dt;
  double isdt = 1.0 / std::sqrt((double)p.dt);
  bool fast = true, rnd = false;
  for (int i = 0; i < TD_T; ++i)
    for (int j = 0; j < TD_T; ++j) {
      int k = i * TD_T + j;
      d.a[k] = p.a[i][j]; d.gamma[k] = p.gamma[i][j]; d.s_R[k] = p.s_R[i][j];
      d.sig[k] = (float)(std::sqrt(2.0 * (double)p.kBT * (double)p.gamma[i][j]) * isdt);
      if (i < p.n_types && j < p.n_types && p.s_R[i][j] != 0.5f) fast = false;
      for (int sp = 0; sp < p.n_species; ++sp) d.kappa[sp][k] = p.kappa[sp][i][j];  // padded species stay 0
    }
  for (int sp = 0; sp < p.n_species; ++sp) {
    d.s_c[sp] = p.s_c[sp];
    d.epsc[sp] = (float)((double)p.m_s[sp] * (double)p.m_s[sp] * (double)p.rho / (double)p.dt);
    d.epsc2[sp] = (float)(-2.0 * std::log(2.0) * (double)p.m_s[sp] * (double)p.m_s[sp] * (double)p.rho / (double)p.dt);
    if (p.s_c[sp] != 2.0f) fast = false;
    if (p.m_s[sp] != 0.0f) rnd = true;
  }
  for (int sp = 0; sp < p.n_species; ++sp)
    for (int t = 0; t < p.n_types; ++t) {
      d.src[sp][t] = p.source[sp][t]; d.dec[sp][t] = p.decay[sp][t];
      if (p.source[sp][t] != 0.0f || p.decay[sp][t] != 0.0f) d.has_source = 1;
    }
  d.body_mode = p.body_mode;
  uint32_t k0 = (uint32_t)(p.seed & 0xffffffffu), k1 = (uint32_t)(p.seed >> 32);
  for (int r = 0; r < 10; ++r) {
    d.key0[r] = k0 + (uint32_t)r * 0x9E3779B9u;
    d.key1[r] = k1 + (uint32_t)r * 0xBB67AE85u;
  }
  d.excl_same = p.exclude_same_cell_membrane_pairs;
  d.fast_w = fast; d.rand_flux = rnd;
}

inline uint32_t spread3(uint32_t v) {  // 10 bits -> every third bit
  uint32_t r = 0;
  for (int b = 0; b < 10; ++b) r |= ((v >> b) & 1u) << (3 * b);
  return r;
}
inline uint32_t morton(uint32_t x, uint32_t y, uint32_t z) { return spread3(x) | (spread3(y) << 1) | (spread3(z) << 2); }

float wrap_host(float x, float L) {
  if (x >= L) x -= L;
  if (x < 0.0f) { x += L; if (x >= L) x = 0.0f; }
  return x;
}

// Derive bonds / dihedrals / per-vertex incidence from a triangle list.  Returns false if the mesh is not a closed,
// consistently oriented manifold.  Bonds are the unique edges (a < b) in lexicographic order; the dihedral of bond
// (a,b) is (c, a, b, d) with triangles (c,a,b) and (d,b,a)  [Eq 19, PAPER.md:124-128].
bool build_template(int nv, int ntri, const int32_t* tri, MeshTemplate& T) {
  std::map<std::pair<int, int>, int> opp;  // directed edge a->b -> third vertex
  for (int t = 0; t < ntri; ++t)
    for (int k = 0; k < 3; ++k) {
      int a = tri[3 * t + k], b = tri[3 * t + (k + 1) % 3], c = tri[3 * t + (k + 2) % 3];
      if (a < 0 || a >= nv || b < 0 || b >= nv || a == b) return false;
      if (!opp.emplace(std::make_pair(a, b), c).second) return false;
    }
  for (auto& kv : opp)
    if (!opp.count({kv.first.second, kv.first.first})) return false;
  T.nv = nv; T.ntri = ntri;
  T.tri.assign(tri, tri + 3 * ntri);
  T.tri16.resize(3 * ntri);
  for (int k = 0; k < 3 * ntri; ++k) T.tri16[k] = (uint16_t)tri[k];
  for (auto& kv : opp) {  // std::map iterates (a,b) lexicographically
    int a = kv.first.first, b = kv.first.second;
    if (a > b) continue;
    T.bond.push_back(a); T.bond.push_back(b);
    T.dih.push_back(kv.second); T.dih.push_back(a); T.dih.push_back(b); T.dih.push_back(opp[{b, a}]);
  }
  T.nbond = (int)T.bond.size() / 2;
  T.dih16.resize(4 * T.nbond);
  for (int k = 0; k < 4 * T.nbond; ++k) T.dih16[k] = (uint16_t)T.dih[k];
  // per-vertex CSR: bonds and triangles share voff (a closed manifold vertex has as many edges as triangles)
  std::vector<std::vector<uint32_t>> vb(nv), vt(nv), vd(nv);
  for (int b = 0; b < T.nbond; ++b) {
    int i = T.bond[2 * b], j = T.bond[2 * b + 1];
    vb[i].push_back((uint32_t)j | ((uint32_t)b << 16));
    vb[j].push_back((uint32_t)i | ((uint32_t)b << 16));
    for (int r = 0; r < 4; ++r) vd[T.dih[4 * b + r]].push_back((uint32_t)b | ((uint32_t)r << 16));
  }
  for (int t = 0; t < ntri; ++t)
    for (int r = 0; r < 3; ++r) vt[tri[3 * t + r]].push_back((uint32_t)t | ((uint32_t)r << 16));
  T.voff.assign(nv + 1, 0); T.vdoff.assign(nv + 1, 0);
  for (int v = 0; v < nv; ++v) {
    if (vb[v].size() != vt[v].size()) return false;
    T.voff[v + 1] = T.voff[v] + (int)vb[v].size();
    T.vdoff[v + 1] = T.vdoff[v] + (int)vd[v].size();
    T.vbond.insert(T.vbond.end(), vb[v].begin(), vb[v].end());
    T.vtri.insert(T.vtri.end(), vt[v].begin(), vt[v].end());
    T.vdih.insert(T.vdih.end(), vd[v].begin(), vd[v].end());
  }
  return true;
}

}  // namespace

// =====================================================================================================
// construction
// =====================================================================================================
extern "C" int tdpd_create(const tdpd_params* p, int device, void* stream_pair, void* stream_bonded, tdpd_sim** out) {
  if (!out) return TDPD_EINVAL;
  *out = nullptr;
  std::string why;
  if (!validate_params(p, why)) return TDPD_EINVAL;
  tdpd_sim* s = new tdpd_sim();
  s->prm = *p;
  derive_params(*p, s->dp);
  s->device = device;
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) { delete s; return TDPD_ECUDA; }
  if (stream_pair && stream_bonded) {
    s->sA = (cudaStream_t)stream_pair; s->sB = (cudaStream_t)stream_bonded;
  } else {
    s->own_streams = true;
    int plo = 0, phi = 0;
    cudaDeviceGetStreamPriorityRange(&plo, &phi);
    if (cudaStreamCreateWithFlags(&s->sA, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithPriority(&s->sB, cudaStreamNonBlocking, phi) != cudaSuccess) { delete s; return TDPD_ECUDA; }
  }
  if (cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming) != cudaSuccess) { delete s; return TDPD_ECUDA; }
  *out = s;
  return TDPD_OK;
}

static int append_particles(tdpd_sim* s, int64_t n, const float* pos, const float* vel, const int32_t* type,
                            int fixed_type, const float* conc, int rbc1) {
  int S = s->prm.n_species;
  for (int64_t i = 0; i < n; ++i) {
    int ty = type ? type[i] : fixed_type;
    if (ty < 0 || ty >= s->prm.n_types) return fail(s, TDPD_EINVAL, "particle type out of range");
  }
  if (s->n + n > 0xFFFFFFF0ll) return fail(s, TDPD_EINVAL, "too many particles");
  for (int64_t i = 0; i < n; ++i) {
    for (int a = 0; a < 3; ++a) {
      s->h_pos.push_back(wrap_host(pos[3 * i + a], s->prm.box[a]));
      s->h_vel.push_back(vel ? vel[3 * i + a] : 0.0f);
    }
    for (int sp = 0; sp < S; ++sp) s->h_conc.push_back(conc ? conc[S * i + sp] : 0.0f);
    s->h_type.push_back(type ? type[i] : fixed_type);
    s->h_rbc.push_back(rbc1);
  }
  s->n += n;
  return TDPD_OK;
}

extern "C" int tdpd_load_particles(tdpd_sim* s, int64_t n, const float* pos, const float* vel, const int32_t* type,
                                   const float* conc) {
  if (!s) return TDPD_EINVAL;
  if (s->finalized) return fail(s, TDPD_ESTATE, "particles cannot be added after tdpd_set_workspace");
  if (n < 0 || (n > 0 && !pos)) return fail(s, TDPD_EINVAL, "bad particle arrays");
  return append_particles(s, n, pos, vel, type, 0, conc, 0);
}

extern "C" int tdpd_add_rbc_mesh(tdpd_sim* s, int32_t nv, const float* verts, const float* vel, const float* conc,
                                 int32_t ntri, const int32_t* tri, const tdpd_rbc_params* rp, int32_t mtype,
                                 int32_t* rbc_index_out) {
  if (!s) return TDPD_EINVAL;
  if (s->finalized) return fail(s, TDPD_ESTATE, "membranes cannot be added after tdpd_set_workspace");
  if (nv < 4 || nv > 4096 || ntri < 4 || ntri > 65535 || !verts || !tri || !rp)
    return fail(s, TDPD_EINVAL, "bad mesh arguments (4 <= nv <= 4096)");
  if (!(rp->p > 0) || !(rp->x0 > 1) || 3.0f * rp->gamma_C < rp->gamma_T || rp->gamma_T < 0)
    return fail(s, TDPD_EINVAL, "bad membrane parameters (need p > 0, x0 > 1, 3 gamma_C >= gamma_T >= 0)");
  if (mtype < 0 || mtype >= s->prm.n_types) return fail(s, TDPD_EINVAL, "membrane type out of range");
  int tmpl = -1;
  for (size_t k = 0; k < s->tmpls.size(); ++k)
    if (s->tmpls[k].nv == nv && s->tmpls[k].ntri == ntri && !memcmp(s->tmpls[k].tri.data(), tri, sizeof(int32_t) * 3 * ntri)) tmpl = (int)k;
  if (tmpl < 0) {
    MeshTemplate T;
    if (!build_template(nv, ntri, tri, T)) return fail(s, TDPD_EINVAL, "mesh is not a closed, consistently oriented manifold");
    if (T.nbond > 65535) return fail(s, TDPD_EINVAL, "too many bonds");
    s->tmpls.push_back(std::move(T));
    tmpl = (int)s->tmpls.size() - 1;
  }
  const MeshTemplate& T = s->tmpls[tmpl];
  RbcHost R;
  R.first_id = s->n; R.tmpl = tmpl; R.nv = nv; R.rp = *rp;
  // unwrap relative to vertex 0 (minimum image), fp64 from the fp32 inputs
  std::vector<double> r(3 * nv);
  for (int v = 0; v < nv; ++v)
    for (int a = 0; a < 3; ++a) {
      double L = s->prm.box[a];
      double x0 = wrap_host(verts[a], s->prm.box[a]), x = wrap_host(verts[3 * v + a], s->prm.box[a]);
      double d = x - x0;
      r[3 * v + a] = x0 + (d - L * std::floor(d / L + 0.5));
    }
  for (int v = 0; v < nv; ++v)
    for (int a = 0; a < 3; ++a)
      if (std::fabs(r[3 * v + a] - r[a]) >= 0.49 * (double)s->prm.box[a])
        return fail(s, TDPD_EINVAL, "membrane extent must stay below half the box (minimum-image unwrap)");
  double kBT = s->prm.kBT, x0r = 1.0 / (double)rp->x0;
  double om = 1.0 - x0r;
  double f0 = kBT / (double)rp->p * (0.25 / (om * om) - 0.25 + x0r);  // dU_WLC/dh at h = h_0 (Eq 13)
  R.h0.resize(T.nbond); R.kp.resize(T.nbond);
  for (int b = 0; b < T.nbond; ++b) {
    int i = T.bond[2 * b], j = T.bond[2 * b + 1];
    double d2 = 0;
    for (int a = 0; a < 3; ++a) { double d = r[3 * i + a] - r[3 * j + a]; d2 += d * d; }
    double h0 = std::sqrt(d2);
    R.h0[b] = (float)h0;
    R.kp[b] = (float)(f0 * std::pow(h0, (double)rp->m));  // force-free at h_0 (R11)
  }
  R.A0t.resize(ntri);
  R.A0 = 0;
  for (int t = 0; t < ntri; ++t) {
    const double *a = &r[3 * tri[3 * t]], *b = &r[3 * tri[3 * t + 1]], *c = &r[3 * tri[3 * t + 2]];
    double u[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]}, w[3] = {c[0] - a[0], c[1] - a[1], c[2] - a[2]};
    double nx = u[1] * w[2] - u[2] * w[1], ny = u[2] * w[0] - u[0] * w[2], nz = u[0] * w[1] - u[1] * w[0];
    double At = 0.5 * std::sqrt(nx * nx + ny * ny + nz * nz);
    R.A0t[t] = (float)At;
    R.A0 += At;
  }
  R.V0 = std::pow(R.A0, 1.5) * (double)rp->VR_over_AR32;
  int rc = append_particles(s, nv, verts, vel, nullptr, mtype, conc, (int)s->rbcs.size() + 1);
  if (rc != TDPD_OK) return rc;
  s->max_nv = std::max(s->max_nv, (int)nv);
  s->rbcs.push_back(std::move(R));
  if (rbc_index_out) *rbc_index_out = (int32_t)s->rbcs.size() - 1;
  return TDPD_OK;
}

// =====================================================================================================
// grid, launch configuration
// =====================================================================================================
static void build_grid(tdpd_sim* s) {
  const int* nc = s->dp.ncell;
  s->ncells = (uint32_t)nc[0] * nc[1] * nc[2];
  s->key_bits = 1;
  while ((1u << s->key_bits) < s->ncells) ++s->key_bits;
  std::vector<std::pair<uint32_t, uint32_t>> codes(s->ncells);  // (morton, linear)
  for (int z = 0; z < nc[2]; ++z)
    for (int y = 0; y < nc[1]; ++y)
      for (int x = 0; x < nc[0]; ++x) {
        uint32_t lin = (uint32_t)((z * nc[1] + y) * nc[0] + x);
        codes[lin] = {morton(x, y, z), lin};
      }
  std::sort(codes.begin(), codes.end());
  s->cell_rank.resize(s->ncells); s->rank_cell.resize(s->ncells);
  for (uint32_t r = 0; r < s->ncells; ++r) {
    uint32_t lin = codes[r].second;
    s->cell_rank[lin] = r;
    uint32_t x = lin % nc[0], y = (lin / nc[0]) % nc[1], z = lin / (nc[0] * nc[1]);
    s->rank_cell[r] = x | (y << 10) | (z << 20);
  }
  // static neighbour runs: the 27 neighbours of a cell, sorted by Morton rank, merged while they are
  // rank-consecutive and share the 2x2x2 block and the periodic image (one displacement per run)
  if (s->seg_off.size() != (size_t)s->ncells + 1) {
    s->seg_off.assign((size_t)s->ncells + 1, 0);
    s->seg_first.clear(); s->seg_meta.clear();
    s->seg_first.reserve((size_t)s->ncells * 14); s->seg_meta.reserve((size_t)s->ncells * 14);
    for (uint32_t r = 0; r < s->ncells; ++r) {
      const uint32_t pc = s->rank_cell[r];
      const int c[3] = {(int)(pc & 1023u), (int)((pc >> 10) & 1023u), (int)(pc >> 20)};
      std::pair<uint32_t, uint64_t> nb[27];  // (rank, signature = block | wrap code << 27)
      for (int k = 0; k < 27; ++k) {
        const int d[3] = {k % 3 - 1, (k / 3) % 3 - 1, k / 9 - 1};
        int q[3];
        uint32_t wcode = 0;
        for (int a = 0; a < 3; ++a) {
          q[a] = c[a] + d[a];
          int w = 0;
          if (q[a] < 0) { q[a] += nc[a]; w = -1; }
          else if (q[a] >= nc[a]) { q[a] -= nc[a]; w = 1; }
          wcode |= (uint32_t)(w + 1) << (2 * a);
        }
        const uint32_t rank = s->cell_rank[(size_t)(q[2] * nc[1] + q[1]) * nc[0] + q[0]];
        const uint32_t blk = (uint32_t)(q[0] >> 1) | ((uint32_t)(q[1] >> 1) << 9) | ((uint32_t)(q[2] >> 1) << 18);
        nb[k] = {rank, (uint64_t)blk | ((uint64_t)wcode << 27)};
      }
      std::sort(nb, nb + 27);
      std::pair<int, std::pair<uint32_t, uint32_t>> runs[27];  // (-cells, (first rank, meta))
      int nr = 0;
      for (int k = 0; k < 27;) {
        int m = 1;
        while (k + m < 27 && m < 15 && nb[k + m].first == nb[k].first + (uint32_t)m && nb[k + m].second == nb[k].second) ++m;
        runs[nr++] = {-m, {nb[k].first, (uint32_t)m | ((uint32_t)(nb[k].second >> 27) << 4)}};
        k += m;
      }
      // longest runs first: every interior cell has the same multiset of run sizes (8, 4, 2, 2, 2, 1 x 9), so the
      // k-th run of all lanes of a warp has the same number of cells and the scan loops stay in step
      std::sort(runs, runs + nr);
      for (int k = 0; k < nr; ++k) {
        s->seg_first.push_back(runs[k].second.first);
        s->seg_meta.push_back(runs[k].second.second);
      }
      s->seg_off[r + 1] = (uint32_t)s->seg_first.size();
    }
  }
  // launch configuration of the pair kernel: NT consecutive slots per CTA; small systems use smaller CTAs so that
  // every SM gets several; the two-ended hit list holds ~1.3 x the mean number of neighbours inside the cutoff
  {
    double rcut = std::max(s->prm.r_c, s->prm.r_cc);
    double mn = 4.18879 * rcut * rcut * rcut * (double)s->n / ((double)s->prm.box[0] * s->prm.box[1] * s->prm.box[2]);
    // sub-wave systems (fewer particles than the GPU has thread slots): several threads per particle
    int split = s->n >= 300000 ? 1 : (s->n >= 20000 ? 2 : 16);
    s->pair_split = s->tune_split ? s->tune_split : split;
    // stack capacity: ~1.9 x the mean number of neighbours (a full stack forces an early, ragged drain), at most 120
    // entries so that three 256-thread CTAs still fit the shared memory of an SM
    int lc = ((int)(mn * 1.9 / s->pair_split) + 8 + 1) / 2 * 2;
    s->lcap = s->tune_lcap ? s->tune_lcap : std::min(120, std::max(16, lc));
    s->pair_nt = s->tune_nt ? s->tune_nt : (s->pair_split <= 2 ? 256 : 128);
    if (s->pair_nt < s->pair_split) s->pair_nt = s->pair_split;
  }
  if (s->nl_skin > 0.0f) {
    // neighbour-list mode: one thread per particle (the list columns are per slot), list capacity ~1.5 x the mean
    // number of particles within cutoff + skin (a full column raises TD_ERR_LIST_OVERFLOW, never overflows)
    double rl = std::max(s->prm.r_c, s->prm.r_cc) + (double)s->nl_skin;
    double mn = 4.18879 * rl * rl * rl * (double)s->n / ((double)s->prm.box[0] * s->prm.box[1] * s->prm.box[2]);
    // next to a membrane both of its sheets add their vertices (surface density nv / A0) inside the list sphere
    double mv = 0.0;
    for (auto& R : s->rbcs) mv = std::max(mv, 2.0 * 3.14159265 * rl * rl * (double)R.nv / R.A0);
    s->nl_cap = s->tune_nl_cap ? s->tune_nl_cap : ((int)(1.5 * mn + 1.25 * mv) + 32 + 7) / 8 * 8;
    s->pair_split = 1;
    s->pair_nt = 256;
    if (!s->tune_lcap) {
      double rcut = std::max(s->prm.r_c, s->prm.r_cc);
      double m0 = 4.18879 * rcut * rcut * rcut * (double)s->n / ((double)s->prm.box[0] * s->prm.box[1] * s->prm.box[2]);
      s->lcap = std::min(120, std::max(16, ((int)(m0 * 1.9) + 8 + 1) / 2 * 2));
    }
  }
  // membrane kernel: CTAs per membrane so that small suspensions still fill the machine
  int M = (int)s->rbcs.size();
  if (M) {
    s->mem_nchunk = std::max(1, std::min(8, (296 + M - 1) / M));
    int CH = (s->max_nv + s->mem_nchunk - 1) / s->mem_nchunk;
    int loops = (CH + 255) / 256;
    s->mem_nt = std::min(256, ((CH + loops - 1) / loops + 31) / 32 * 32);
  }
}

struct Carver {
  unsigned char* base;
  size_t off = 0;
  template <class T> T* take(size_t count) {
    off = (off + 255) & ~(size_t)255;
    T* p = base ? (T*)(base + off) : nullptr;
    off += count * sizeof(T);
    return p;
  }
};

// assigns every device array inside the workspace (base may be NULL: size query only); returns bytes
static size_t layout(tdpd_sim* s, void* basep) {
  Carver c{(unsigned char*)basep};
  size_t n = (size_t)std::max<int64_t>(s->n, 1);
  int S = s->prm.n_species;
  for (int k = 0; k < 2; ++k) {
    s->st[k].pos = c.take<float4>(n);
    s->st[k].vel = c.take<float4>(n);
    s->st[k].cx = c.take<float>(n * (size_t)std::max(S - 1, 1));
    s->st[k].lo = c.take<float4>(n);
    s->keys[k] = c.take<uint32_t>(n);
    s->vals[k] = c.take<uint32_t>(n);
  }
  s->sort_scratch = c.take<unsigned char>(td_sort_scratch_bytes((int64_t)n));
  s->cell_start = c.take<uint32_t>(s->ncells + 1);
  s->cell_rank_d = c.take<uint32_t>(s->ncells);
  s->rank_cell_d = c.take<uint32_t>(s->ncells);
  s->seg_off_d = c.take<uint32_t>(s->seg_off.size());
  s->seg_first_d = c.take<uint32_t>(s->seg_first.size());
  s->seg_meta_d = c.take<uint32_t>(s->seg_meta.size());
  s->rec.P4 = c.take<float4>(n);
  s->rec.R8 = c.take<float4>(2 * n);
  s->rec.Y4 = c.take<float4>(std::max<size_t>(1, n * (size_t)td_species_groups(S)));
  s->slot_of_id = c.take<uint32_t>(n);
  s->F4 = c.take<float4>(n);
  s->Fb = c.take<float4>(n);
  s->Qx = c.take<float>(n * (size_t)std::max(S - 1, 1));
  s->staging = c.take<float>(n * (size_t)(9 + 2 * std::max(S, 4)));  // id-ordered pos, vel, force [n][3], conc, flux [n][S]
  s->err_d = c.take<int>(64);
  s->step_d = c.take<uint32_t>(64);
  if (s->nl_skin > 0.0f) {
    s->okey_d = c.take<uint32_t>(n);
    s->P4ref_d = c.take<float4>(n);
    s->nl_cnt_d = c.take<uint32_t>(n);
    s->nlist_d = c.take<uint16_t>(((n + 255) / 256) * (size_t)s->nl_cap * 256);
  }
  size_t M = s->rbcs.size();
  s->stats_d = c.take<double>(4 * std::max<size_t>(M, 1));  // two slots (step parity) of (area, volume) per membrane
  s->rbcs_d = c.take<RbcDev>(std::max<size_t>(M, 1));
  s->tmpls_d = c.take<MeshTemplateDev>(std::max<size_t>(s->tmpls.size(), 1));
  size_t nb = 0, nt = 0, topo = 0;
  for (auto& R : s->rbcs) { nb += R.h0.size(); nt += R.A0t.size(); }
  for (auto& T : s->tmpls)
    topo += 256 * 8 + T.tri16.size() * 2 + T.dih16.size() * 2 + (T.voff.size() + T.vdoff.size()) * 4 +
            (T.vbond.size() + T.vtri.size() + T.vdih.size()) * 4;
  s->h0_d = c.take<float>(std::max<size_t>(nb, 1));
  s->kp_d = c.take<float>(std::max<size_t>(nb, 1));
  s->A0t_d = c.take<float>(std::max<size_t>(nt, 1));
  s->topo_d = c.take<unsigned char>(std::max<size_t>(topo, 1));
  return (c.off + 255) & ~(size_t)255;
}

extern "C" int tdpd_workspace_bytes(const tdpd_sim* cs, size_t* bytes) {
  tdpd_sim* s = const_cast<tdpd_sim*>(cs);
  if (!s || !bytes) return TDPD_EINVAL;
  if (s->finalized) { *bytes = s->ws_bytes; return TDPD_OK; }
  build_grid(s);
  *bytes = layout(s, nullptr);
  return TDPD_OK;
}

extern "C" int tdpd_set_workspace(tdpd_sim* s, void* dev_ptr, size_t bytes) {
  if (!s) return TDPD_EINVAL;
  if (s->finalized) return fail(s, TDPD_ESTATE, "workspace already set");
  CK(cudaSetDevice(s->device));
  build_grid(s);
  size_t need = layout(s, nullptr);
  if (dev_ptr) {
    if (bytes < need) return fail(s, TDPD_ENOMEM, "workspace too small");
    if (((uintptr_t)dev_ptr & 255) != 0) return fail(s, TDPD_EINVAL, "workspace must be 256-byte aligned");
    s->ws = dev_ptr;
  } else {
    if (cudaMalloc(&s->ws, need) != cudaSuccess) return fail(s, TDPD_ENOMEM, "cudaMalloc of the workspace failed");
    s->own_ws = true;
  }
  {  // list entries address a candidate by an 11-bit offset inside a run of up to 8 (15 at most) cells
    const double per_run = 8.0 * (double)s->n / std::max<double>(1.0, (double)s->ncells);
    if (per_run > 1400.0)
      return fail(s, TDPD_EINVAL, "more than ~175 particles per cell on average: a run of neighbour cells would exceed the 2047 "
                                  "candidates a list entry can address (use a smaller cutoff-to-density ratio)");
  }
  s->ws_bytes = need;
  layout(s, s->ws);
  const int64_t n = s->n;
  const int S = s->prm.n_species;
  cudaStream_t q = s->sA;
  CK(cudaMemsetAsync(s->ws, 0, need, q));
  // particle state in id order = initial "sorted" side 0
  {
    std::vector<float4> hp(n), hv(n), hm(n);
    std::vector<float> hc((size_t)std::max(S - 1, 1) * std::max<int64_t>(n, 1));
    for (int64_t i = 0; i < n; ++i) {
      uint32_t idb = (uint32_t)i;
      float idf;
      memcpy(&idf, &idb, 4);
      hp[i] = make_float4(s->h_pos[3 * i], s->h_pos[3 * i + 1], s->h_pos[3 * i + 2], idf);
      hv[i] = make_float4(s->h_vel[3 * i], s->h_vel[3 * i + 1], s->h_vel[3 * i + 2], s->h_conc[(size_t)S * i]);
      uint32_t mb = td_meta(s->h_type[i], s->h_rbc[i]);
      float mf;
      memcpy(&mf, &mb, 4);
      hm[i] = make_float4(0.f, 0.f, 0.f, mf);
      for (int sp = 1; sp < S; ++sp) hc[(size_t)(sp - 1) * n + i] = s->h_conc[(size_t)S * i + sp];
    }
    if (n) {
      CK(cudaMemcpyAsync(s->st[0].pos, hp.data(), n * sizeof(float4), cudaMemcpyHostToDevice, q));
      CK(cudaMemcpyAsync(s->st[0].vel, hv.data(), n * sizeof(float4), cudaMemcpyHostToDevice, q));
      CK(cudaMemcpyAsync(s->st[0].lo, hm.data(), n * sizeof(float4), cudaMemcpyHostToDevice, q));
      if (S > 1) CK(cudaMemcpyAsync(s->st[0].cx, hc.data(), (size_t)(S - 1) * n * sizeof(float), cudaMemcpyHostToDevice, q));
    }
    CK(cudaStreamSynchronize(q));
  }
  CK(cudaMemcpyAsync(s->cell_rank_d, s->cell_rank.data(), s->ncells * 4, cudaMemcpyHostToDevice, q));
  CK(cudaMemcpyAsync(s->rank_cell_d, s->rank_cell.data(), s->ncells * 4, cudaMemcpyHostToDevice, q));
  CK(cudaMemcpyAsync(s->seg_off_d, s->seg_off.data(), s->seg_off.size() * 4, cudaMemcpyHostToDevice, q));
  CK(cudaMemcpyAsync(s->seg_first_d, s->seg_first.data(), s->seg_first.size() * 4, cudaMemcpyHostToDevice, q));
  CK(cudaMemcpyAsync(s->seg_meta_d, s->seg_meta.data(), s->seg_meta.size() * 4, cudaMemcpyHostToDevice, q));
  // membranes
  std::vector<MeshTemplateDev> td(s->tmpls.size());
  std::vector<unsigned char> topo;
  auto put = [&](const void* src, size_t bytes_) -> size_t {
    size_t o = (topo.size() + 255) & ~(size_t)255;
    topo.resize(o + bytes_);
    memcpy(topo.data() + o, src, bytes_);
    return o;
  };
  for (size_t k = 0; k < s->tmpls.size(); ++k) {
    const MeshTemplate& T = s->tmpls[k];
    td[k].nv = T.nv; td[k].ntri = T.ntri; td[k].nbond = T.nbond;
    td[k].tri = (const uint16_t*)(s->topo_d + put(T.tri16.data(), T.tri16.size() * 2));
    td[k].dih = (const uint16_t*)(s->topo_d + put(T.dih16.data(), T.dih16.size() * 2));
    td[k].voff = (const int*)(s->topo_d + put(T.voff.data(), T.voff.size() * 4));
    td[k].vbond = (const uint32_t*)(s->topo_d + put(T.vbond.data(), T.vbond.size() * 4));
    td[k].vtri = (const uint32_t*)(s->topo_d + put(T.vtri.data(), T.vtri.size() * 4));
    td[k].vdoff = (const int*)(s->topo_d + put(T.vdoff.data(), T.vdoff.size() * 4));
    td[k].vdih = (const uint32_t*)(s->topo_d + put(T.vdih.data(), T.vdih.size() * 4));
  }
  std::vector<RbcDev> rd(s->rbcs.size());
  std::vector<float> h0, kp, a0t;
  double kBT = s->prm.kBT, pre = std::sqrt(2.0 * kBT / (double)s->prm.dt);
  for (size_t m = 0; m < s->rbcs.size(); ++m) {
    const RbcHost& R = s->rbcs[m];
    RbcDev& D = rd[m];
    D.first_id = R.first_id; D.tmpl = R.tmpl;
    D.data_off = (int)h0.size(); D.tri_off = (int)a0t.size();
    h0.insert(h0.end(), R.h0.begin(), R.h0.end());
    kp.insert(kp.end(), R.kp.begin(), R.kp.end());
    a0t.insert(a0t.end(), R.A0t.begin(), R.A0t.end());
    D.A0 = R.A0; D.V0 = R.V0;
    D.kBT_over_p = (float)(kBT / (double)R.rp.p);
    D.inv_x0 = (float)(1.0 / (double)R.rp.x0);
    D.m_pow = R.rp.m; D.gamma_T = R.rp.gamma_T; D.gamma_C = R.rp.gamma_C;
    D.k_g = R.rp.k_g; D.k_l = R.rp.k_l; D.k_v = R.rp.k_v; D.k_b = R.rp.k_b;
    D.cos_t0 = (float)std::cos((double)R.rp.theta0); D.sin_t0 = (float)std::sin((double)R.rp.theta0);
    D.rnd_T = (float)(pre * std::sqrt(2.0 * (double)R.rp.gamma_T));
    D.rnd_C = (float)(pre * std::sqrt(std::max(0.0, 3.0 * (double)R.rp.gamma_C - (double)R.rp.gamma_T)) / 3.0);
  }
  if (!rd.empty()) {
    CK(cudaMemcpyAsync(s->topo_d, topo.data(), topo.size(), cudaMemcpyHostToDevice, q));
    CK(cudaMemcpyAsync(s->tmpls_d, td.data(), td.size() * sizeof(MeshTemplateDev), cudaMemcpyHostToDevice, q));
    CK(cudaMemcpyAsync(s->rbcs_d, rd.data(), rd.size() * sizeof(RbcDev), cudaMemcpyHostToDevice, q));
    CK(cudaMemcpyAsync(s->h0_d, h0.data(), h0.size() * 4, cudaMemcpyHostToDevice, q));
    CK(cudaMemcpyAsync(s->kp_d, kp.data(), kp.size() * 4, cudaMemcpyHostToDevice, q));
    CK(cudaMemcpyAsync(s->A0t_d, a0t.data(), a0t.size() * 4, cudaMemcpyHostToDevice, q));
  }
  CK(cudaStreamSynchronize(q));
  s->h_pos.clear(); s->h_pos.shrink_to_fit(); s->h_vel.clear(); s->h_vel.shrink_to_fit();
  s->h_conc.clear(); s->h_conc.shrink_to_fit(); s->h_type.clear(); s->h_rbc.clear();
  s->finalized = true; s->cur = 0; s->binned = false; s->have_forces = false; s->step = 0;
  return TDPD_OK;
}

// =====================================================================================================
// step orchestration
// =====================================================================================================
namespace {
void drop_graphs(tdpd_sim* s);
struct Scope {  // optional event pair around a group of launches on one stream
  tdpd_sim* s; int cls; cudaStream_t q; cudaEvent_t e1 = nullptr;
  Scope(tdpd_sim* s_, int cls_, cudaStream_t q_) : s(s_), cls(cls_), q(q_) {
    if (s->timing) {
      cudaEvent_t e0;
      cudaEventCreate(&e0); cudaEventCreate(&e1);
      cudaEventRecord(e0, q);
      s->timers[cls].ev.push_back({e0, e1});
    }
  }
  ~Scope() { if (e1) cudaEventRecord(e1, q); }
};

PairArgs pair_args(tdpd_sim* s, int c) {
  PairArgs A;
  A.rec = s->rec; A.vel = s->st[c].vel; A.pos = s->st[c].pos; A.lo = s->st[c].lo;
  A.keys = s->nl_skin > 0.0f ? s->okey_d : s->keys_sorted;
  A.cell_start = s->cell_start; A.cell_rank = s->cell_rank_d; A.rank_cell = s->rank_cell_d;
  A.seg_off = s->seg_off_d; A.seg_first = s->seg_first_d; A.seg_meta = s->seg_meta_d;
  A.F4 = s->F4; A.Qx = s->Qx; A.n = s->n; A.step_p = s->step_d; A.lcap = s->lcap; A.err = s->err_d;
  A.nlist = s->nlist_d; A.nl_cnt = s->nl_cnt_d; A.nl_cap = s->nl_cap;
  const float rl = std::max(s->prm.r_c, s->prm.r_cc) + s->nl_skin;
  A.rlist2 = rl * rl;
  A.census = nullptr;
  return A;
}

int bin_and_sort(tdpd_sim* s, int mode /*0 keys only, 1 open, 2 close+open*/) {
  const bool lm = s->nl_skin > 0.0f;
  const int c = s->cur;  // neighbour-list mode: always side 0
  ListRefresh LR = {s->okey_d, s->rank_cell_d, s->rec, s->P4ref_d};
  {
    Scope t(s, 0, s->sA);
    if (mode == 0) td_launch_init_keys(s->dp, s->st[c], s->n, s->keys[0], s->vals[0], s->cell_rank_d, s->sA);
    else td_launch_kick_drift_key(s->dp, s->st[c], s->F4, s->Qx, s->Fb, s->n, s->keys[0], s->vals[0], s->cell_rank_d,
                                  mode == 2, s->step_d, lm ? &LR : nullptr, s->sA);
    s->launches += 1; s->timers[0].launches += 1;
  }
  const uint32_t* gate = nullptr;
  if (lm) {  // the device decides whether this step re-bins; the binning kernels below return at once if not
    Scope t(s, 6, s->sA);
    if (mode == 0) {  // first evaluation / after set_state: positions are new, bin unconditionally
      static const uint32_t one = 1u;
      CK(cudaMemcpyAsync(s->step_d + TD_CTL_FORCE, &one, 4, cudaMemcpyHostToDevice, s->sA));
    }
    td_launch_list_decide(s->step_d, s->nl_skin * s->nl_skin, s->sA);
    s->launches += 1; s->timers[6].launches += 1;
    gate = s->step_d;
  }
  int side, nl = 0;
  {
    Scope t(s, 1, s->sA);
    side = td_launch_sort(s->keys, s->vals, s->n, s->key_bits, s->sort_scratch, s->sA, &nl, gate);
    s->launches += nl; s->timers[1].launches += nl;
  }
  {
    Scope t(s, 2, s->sA);
    td_launch_reorder(s->dp, s->st[c], s->st[c ^ 1], s->rec, s->keys[side], s->vals[side], s->rank_cell_d, s->n,
                      s->ncells, s->cell_start, s->slot_of_id, lm ? s->okey_d : nullptr, s->P4ref_d, gate, s->sA);
    s->keys_sorted = s->keys[side];
    s->launches += 1; s->timers[2].launches += 1;
    if (lm && s->n) {  // the state stays on side 0
      td_launch_copy_state(s->dp, s->st[c ^ 1], s->st[c], s->n, gate, s->sA);
      s->launches += 1; s->timers[2].launches += 1;
    }
  }
  if (lm) {
    Scope t(s, 6, s->sA);
    int rc = td_launch_build_list(s->dp, pair_args(s, c), gate, s->sA);
    if (rc) return fail(s, TDPD_ECUDA, std::string("list kernel attribute: ") + cudaGetErrorString((cudaError_t)rc));
    if (s->n) { s->launches += 1; s->timers[6].launches += 1; }
  } else {
    s->cur = c ^ 1;
  }
  s->binned = true;
  CK(cudaGetLastError());
  return TDPD_OK;
}

int eval_forces(tdpd_sim* s) {
  const int c = s->cur;
  const bool mem = !s->rbcs.empty();
  // the membrane kernel (stream B) is enqueued BEFORE the pair kernel: its few CTAs take their SM slots at once and
  // the pair grid fills the rest; enqueued after it, they only got slots as the pair grid drained (0.15 ms of the
  // step in round 1).  The binding also gives stream B the higher priority.
  if (mem) {
    CK(cudaEventRecord(s->ev_fork, s->sA));
    CK(cudaStreamWaitEvent(s->sB, s->ev_fork, 0));
    {
      Scope t(s, 4, s->sB);
      MembraneArgs M;
      M.st = s->st[c]; M.slot_of_id = s->slot_of_id; M.rbcs = s->rbcs_d; M.tmpls = s->tmpls_d;
      M.h0 = s->h0_d; M.kp = s->kp_d; M.A0t = s->A0t_d; M.Fb = s->Fb; M.stats = s->stats_d;
      M.nchunk = s->mem_nchunk; M.step_p = s->step_d; M.err = s->err_d; M.lag_av = s->lag_av ? 1 : 0;
      int rc = td_launch_membrane(s->dp, M, (int)s->rbcs.size(), s->max_nv, s->mem_nt, s->sB);
      if (rc) return fail(s, TDPD_ECUDA, std::string("membrane kernel attribute: ") + cudaGetErrorString((cudaError_t)rc));
      s->launches += 1; s->timers[4].launches += 1;
    }
    CK(cudaEventRecord(s->ev_join, s->sB));
  }
  {
    Scope t(s, 3, s->sA);
    int rc = td_launch_pair(s->dp, pair_args(s, c), s->pair_nt, s->pair_split, s->nl_skin > 0.0f, s->sA);
    if (rc) return fail(s, TDPD_ECUDA, std::string("pair kernel attribute: ") + cudaGetErrorString((cudaError_t)rc));
    s->launches += 1; s->timers[3].launches += 1;
  }
  if (mem) CK(cudaStreamWaitEvent(s->sA, s->ev_join, 0));
  CK(cudaGetLastError());
  s->have_forces = true;
  return TDPD_OK;
}

int ensure_forces(tdpd_sim* s) {
  if (!s->finalized) return fail(s, TDPD_ESTATE, "tdpd_set_workspace has not been called");
  CK(cudaSetDevice(s->device));
  if (s->have_forces) return TDPD_OK;
  // always re-bin: the reorder kernel also refreshes the pair kernel's records (concentrations, positions)
  { int rc = bin_and_sort(s, 0); if (rc) return rc; }
  return eval_forces(s);
}
}  // namespace

namespace {
// enqueues one velocity-Verlet step: opening half-kick (fused with the closing one of the previous step of this call),
// drift, binning, forces, and the closing half-kick if this is the last step of the call
int enqueue_step(tdpd_sim* s, bool first, bool last) {
  int rc = bin_and_sort(s, first ? 1 : 2);
  if (rc) return rc;
  rc = eval_forces(s);
  if (rc) return rc;
  if (last) {
    Scope t(s, 5, s->sA);
    td_launch_kick(s->dp, s->st[s->cur], s->F4, s->Qx, s->Fb, s->n, s->sA);
    s->launches += 1; s->timers[5].launches += 1;
  }
  CK(cudaGetLastError());
  return TDPD_OK;
}

void drop_graphs(tdpd_sim* s) {
  for (auto& a : s->gexec) for (auto& b : a) for (auto& g : b) { if (g) cudaGraphExecDestroy(g); g = nullptr; }
}
}  // namespace

extern "C" int tdpd_step(tdpd_sim* s, int32_t nsteps) {
  if (!s) return TDPD_EINVAL;
  if (nsteps < 0) return fail(s, TDPD_EINVAL, "nsteps < 0");
  int rc = ensure_forces(s);
  if (rc || nsteps == 0) return rc;
  for (int32_t it = 0; it < nsteps; ++it) {
    const bool first = it == 0, last = it == nsteps - 1;
    s->step += 1;  // the integrator bumps the device copy
    if (!s->use_graph || s->timing || s->n == 0) {
      if ((rc = enqueue_step(s, first, last))) return rc;
      continue;
    }
    // one CUDA graph per (ping-pong side, first, last): the launch sequence of a step is static, and the step word
    // lives in device memory, so replaying the graph is all a step needs
    const int side = s->cur;
    cudaGraphExec_t& ge = s->gexec[side][first][last];
    if (!ge) {
      const int64_t l0 = s->launches;
      cudaGraph_t g = nullptr;
      bool ok = cudaStreamBeginCapture(s->sA, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
      if (ok) {
        rc = enqueue_step(s, first, last);
        ok = cudaStreamEndCapture(s->sA, &g) == cudaSuccess && rc == TDPD_OK && g;
        ok = ok && cudaGraphInstantiate(&ge, g, 0) == cudaSuccess;
        if (g) cudaGraphDestroy(g);
      }
      if (!ok) {  // capture is not available here: fall back to plain launches for good
        cudaGetLastError();
        ge = nullptr;
        s->use_graph = false;
        drop_graphs(s);
        s->cur = side;
        if ((rc = enqueue_step(s, first, last))) return rc;
        continue;
      }
      s->glaunches[side][first][last] = (int)(s->launches - l0);
      s->gkeys[side][first][last] = s->keys_sorted;
      s->launches = l0;  // counted at launch below
      s->cur = side;     // the capture advanced the host bookkeeping; the launch below does it again
    }
    CK(cudaGraphLaunch(ge, s->sA));
    s->cur = s->nl_skin > 0.0f ? side : side ^ 1;  // neighbour-list mode keeps the state on one side
    s->keys_sorted = s->gkeys[side][first][last];
    s->launches += s->glaunches[side][first][last];
    s->binned = true; s->have_forces = true;
  }
  return TDPD_OK;
}

extern "C" int tdpd_sync(tdpd_sim* s) {
  if (!s) return TDPD_EINVAL;
  CK(cudaSetDevice(s->device));
  CK(cudaStreamSynchronize(s->sA));
  CK(cudaStreamSynchronize(s->sB));
  return TDPD_OK;
}

// =====================================================================================================
// read-back
// =====================================================================================================
static int check_err_word(tdpd_sim* s) {
  int w = 0;
  CK(cudaMemcpy(&w, s->err_d, sizeof w, cudaMemcpyDeviceToHost));
  if (w) {
    int zero = 0;
    cudaMemcpy(s->err_d, &zero, sizeof zero, cudaMemcpyHostToDevice);
    std::string m;
    if (w & TD_ERR_CELL_OVERFLOW) m += "pair kernel: a run of neighbour cells (up to 8 cells) holds more than 2047 particles; ";
    if (w & TD_ERR_LIST_OVERFLOW) m += "neighbour list: a particle has more neighbours within cutoff + skin than the list capacity (raise list_cap in tdpd_set_neighbor_list); ";
    if (w & TD_ERR_NONFINITE) m += "non-finite value in the state; ";
    if (w & TD_ERR_BOND_OVERSTRETCH) m += "a WLC bond reached x >= 1; ";
    return fail(s, TDPD_EUNSTABLE, m);
  }
  return TDPD_OK;
}

// id-ordered read-back: every requested array is unsorted into its own part of the staging area and copied out
// asynchronously; ONE stream synchronisation at the end (round 1: one kernel + one blocking copy + one sync per array)
static int fetch_begin(tdpd_sim* s, int what, int width, float* host, size_t& off) {
  if (!host || s->n == 0) return TDPD_OK;
  float* dst = s->staging + off;
  off += (size_t)s->n * width;
  td_launch_unsort(s->st[s->cur], s->F4, s->Qx, s->Fb, s->n, s->prm.n_species, what, dst, s->err_d, s->dp.box, s->sA);
  s->launches += 1;
  CK(cudaMemcpyAsync(host, dst, (size_t)s->n * width * sizeof(float), cudaMemcpyDeviceToHost, s->sA));
  return TDPD_OK;
}

extern "C" int tdpd_get_state(tdpd_sim* s, float* pos, float* vel, float* conc, float* force, float* flux,
                              int64_t* step) {
  if (!s) return TDPD_EINVAL;
  if (!s->finalized) return fail(s, TDPD_ESTATE, "tdpd_set_workspace has not been called");
  int rc;
  if (force || flux) { rc = ensure_forces(s); if (rc) return rc; }
  CK(cudaSetDevice(s->device));
  const int S = s->prm.n_species;
  size_t off = 0;
  if ((rc = fetch_begin(s, 0, 3, pos, off))) return rc;
  if ((rc = fetch_begin(s, 1, 3, vel, off))) return rc;
  if ((rc = fetch_begin(s, 2, S, conc, off))) return rc;
  if ((rc = fetch_begin(s, 3, 3, force, off))) return rc;
  if ((rc = fetch_begin(s, 4, S, flux, off))) return rc;
  if ((rc = tdpd_sync(s))) return rc;
  if (step) *step = s->step;
  return check_err_word(s);
}

extern "C" int tdpd_get_forces_split(tdpd_sim* s, float* force_pair, float* force_bonded) {
  if (!s) return TDPD_EINVAL;
  int rc = ensure_forces(s);
  if (rc) return rc;
  size_t off = 0;
  if ((rc = fetch_begin(s, 5, 3, force_pair, off))) return rc;
  if ((rc = fetch_begin(s, 6, 3, force_bonded, off))) return rc;
  if ((rc = tdpd_sync(s))) return rc;
  return check_err_word(s);
}

extern "C" int64_t tdpd_num_particles(const tdpd_sim* s) { return s ? s->n : 0; }
extern "C" int32_t tdpd_num_rbc(const tdpd_sim* s) { return s ? (int32_t)s->rbcs.size() : 0; }

extern "C" int tdpd_get_rbc_stats(tdpd_sim* s, double* area, double* volume, double* A0, double* V0) {
  if (!s) return TDPD_EINVAL;
  size_t M = s->rbcs.size();
  if (area || volume) {
    int rc = ensure_forces(s);
    if (rc) return rc;
    if ((rc = tdpd_sync(s))) return rc;
    std::vector<double> st(2 * std::max<size_t>(M, 1));
    if (M) CK(cudaMemcpy(st.data(), s->stats_d + (size_t)(s->step & 1) * 2 * M, 2 * M * sizeof(double), cudaMemcpyDeviceToHost));
    for (size_t m = 0; m < M; ++m) {
      if (area) area[m] = st[2 * m];
      if (volume) volume[m] = st[2 * m + 1];
    }
  }
  for (size_t m = 0; m < M; ++m) {
    if (A0) A0[m] = s->rbcs[m].A0;
    if (V0) V0[m] = s->rbcs[m].V0;
  }
  return TDPD_OK;
}

extern "C" int tdpd_get_rbc_topology(tdpd_sim* s, int32_t m, int32_t* nbond, int32_t* bond, int32_t* dih, float* h0,
                                     float* kp, float* A0t) {
  if (!s || m < 0 || m >= (int32_t)s->rbcs.size()) return TDPD_EINVAL;
  const RbcHost& R = s->rbcs[m];
  const MeshTemplate& T = s->tmpls[R.tmpl];
  if (nbond) *nbond = T.nbond;
  if (bond) memcpy(bond, T.bond.data(), T.bond.size() * 4);
  if (dih) memcpy(dih, T.dih.data(), T.dih.size() * 4);
  if (h0) memcpy(h0, R.h0.data(), R.h0.size() * 4);
  if (kp) memcpy(kp, R.kp.data(), R.kp.size() * 4);
  if (A0t) memcpy(A0t, R.A0t.data(), R.A0t.size() * 4);
  return TDPD_OK;
}

extern "C" int tdpd_set_params(tdpd_sim* s, const tdpd_params* p) {
  if (!s) return TDPD_EINVAL;
  std::string why;
  if (!validate_params(p, why)) return fail(s, TDPD_EINVAL, why);
  DevParams d;
  derive_params(*p, d, s->nl_skin);
  if (s->finalized) {
    if (p->n_types != s->prm.n_types || p->n_species != s->prm.n_species ||
        memcmp(d.ncell, s->dp.ncell, sizeof d.ncell) || memcmp(d.box, s->dp.box, sizeof d.box))
      return fail(s, TDPD_EINVAL, "box, cell grid and type/species counts are fixed after tdpd_set_workspace");
    if (!s->rbcs.empty() && (p->kBT != s->prm.kBT || p->dt != s->prm.dt))
      return fail(s, TDPD_EINVAL, "kBT and dt are fixed after tdpd_set_workspace when membranes are present");
  } else {
    if ((p->n_types != s->prm.n_types || p->n_species != s->prm.n_species) && s->n)
      return fail(s, TDPD_EINVAL, "type/species counts cannot change once particles are loaded");
    // k_p, h_0, A_0, V_0 of a loaded membrane were derived from kBT and the box at tdpd_add_rbc_mesh
    if (!s->rbcs.empty() && (p->kBT != s->prm.kBT || p->dt != s->prm.dt || memcmp(p->box, s->prm.box, sizeof p->box)))
      return fail(s, TDPD_EINVAL, "kBT, dt and box are fixed once a membrane is loaded");
  }
  s->prm = *p;
  s->dp = d;
  s->have_forces = false;
  drop_graphs(s);  // the parameters are baked into the captured kernel nodes
  return TDPD_OK;
}

extern "C" int tdpd_set_state(tdpd_sim* s, const float* pos, const float* vel, const float* conc) {
  if (!s) return TDPD_EINVAL;
  if (!s->finalized) return fail(s, TDPD_ESTATE, "tdpd_set_workspace has not been called");
  CK(cudaSetDevice(s->device));
  int rc = tdpd_sync(s);
  if (rc) return rc;
  const size_t n = (size_t)s->n;
  const int S = s->prm.n_species;
  float *dpos = nullptr, *dvel = nullptr, *dconc = nullptr;
  if (pos) { dpos = s->staging; CK(cudaMemcpyAsync(dpos, pos, n * 3 * 4, cudaMemcpyHostToDevice, s->sA)); }
  if (vel) { dvel = s->staging + n * 4; CK(cudaMemcpyAsync(dvel, vel, n * 3 * 4, cudaMemcpyHostToDevice, s->sA)); }
  if (conc) { dconc = s->staging + n * 8; CK(cudaMemcpyAsync(dconc, conc, n * S * 4, cudaMemcpyHostToDevice, s->sA)); }
  td_launch_set_state(s->dp, s->st[s->cur], s->n, dpos, dvel, dconc, s->sA);
  s->launches += 1;
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(s->sA));  // the caller's buffers are free again when this returns
  if (pos) s->binned = false;
  s->have_forces = false;
  CK(cudaMemsetAsync(s->step_d + TD_CTL_LAGOK, 0, 4, s->sA));  // the membrane totals of the previous step are void
  return TDPD_OK;
}

// =====================================================================================================
// debug / test support
// =====================================================================================================
extern "C" int tdpd_debug_get_binning(tdpd_sim* s, int32_t* cell_xyz, int32_t ncell[3], int32_t* cell_count,
                                      int32_t* sorted_id) {
  if (!s) return TDPD_EINVAL;
  if (s->nl_skin > 0.0f) s->have_forces = false;  // neighbour-list mode: the slots may be those of an older binning
  int rc = ensure_forces(s);
  if (rc) return rc;
  if ((rc = tdpd_sync(s))) return rc;
  if (ncell) for (int a = 0; a < 3; ++a) ncell[a] = s->dp.ncell[a];
  if (!cell_xyz) return TDPD_OK;
  size_t n = (size_t)s->n;
  int32_t *d_xyz = nullptr, *d_cnt = nullptr, *d_sid = nullptr;
  CK(cudaMalloc(&d_xyz, std::max<size_t>(n, 1) * 12));
  CK(cudaMalloc(&d_cnt, (size_t)s->ncells * 4));
  CK(cudaMalloc(&d_sid, std::max<size_t>(n, 1) * 4));
  CK(cudaMemsetAsync(d_cnt, 0, (size_t)s->ncells * 4, s->sA));
  td_launch_binning_debug(s->dp, s->st[s->cur], s->n, s->nl_skin > 0.0f ? s->okey_d : s->keys_sorted, s->rank_cell_d, d_xyz, d_cnt, d_sid, s->sA);
  s->launches += 1;
  CK(cudaMemcpyAsync(cell_xyz, d_xyz, n * 12, cudaMemcpyDeviceToHost, s->sA));
  if (cell_count) CK(cudaMemcpyAsync(cell_count, d_cnt, (size_t)s->ncells * 4, cudaMemcpyDeviceToHost, s->sA));
  if (sorted_id) CK(cudaMemcpyAsync(sorted_id, d_sid, n * 4, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaStreamSynchronize(s->sA));
  cudaFree(d_xyz); cudaFree(d_cnt); cudaFree(d_sid);
  return TDPD_OK;
}

extern "C" int tdpd_debug_neighbor_census(tdpd_sim* s, int32_t* n_rc, int32_t* n_rcc, uint32_t* xor_rc,
                                          uint32_t* xor_rcc) {
  if (!s || !n_rc || !n_rcc || !xor_rc || !xor_rcc) return TDPD_EINVAL;
  if (s->nl_skin > 0.0f) s->have_forces = false;  // re-bin: the census walks the cell table
  int rc = ensure_forces(s);
  if (rc) return rc;
  if ((rc = tdpd_sync(s))) return rc;
  size_t n = std::max<size_t>((size_t)s->n, 1);
  int32_t* d = nullptr;
  CK(cudaMalloc(&d, n * 16));
  td_launch_census(s->dp, s->st[s->cur], s->cell_start, s->cell_rank_d, s->nl_skin > 0.0f ? s->okey_d : s->keys_sorted, s->rank_cell_d, s->n, d, d + n, (uint32_t*)(d + 2 * n),
                   (uint32_t*)(d + 3 * n), s->sA);
  s->launches += 1;
  size_t b = (size_t)s->n * 4;
  CK(cudaMemcpyAsync(n_rc, d, b, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaMemcpyAsync(n_rcc, d + n, b, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaMemcpyAsync(xor_rc, d + 2 * n, b, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaMemcpyAsync(xor_rcc, d + 3 * n, b, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaStreamSynchronize(s->sA));
  cudaFree(d);
  return TDPD_OK;
}

extern "C" int tdpd_debug_pair_census(tdpd_sim* s, int32_t* n_front, int32_t* n_ring, uint32_t* xor_front,
                                      uint32_t* xor_ring) {
  if (!s || !n_front || !n_ring || !xor_front || !xor_ring) return TDPD_EINVAL;
  int rc = ensure_forces(s);   // the binning (and, in list mode, the list) the pair kernel works on
  if (rc) return rc;
  if ((rc = tdpd_sync(s))) return rc;
  if (s->n == 0) return TDPD_OK;
  const size_t n = (size_t)s->n;
  uint32_t* d = nullptr;
  CK(cudaMalloc(&d, n * 16));
  CK(cudaMemsetAsync(d, 0, n * 16, s->sA));
  PairArgs A = pair_args(s, s->cur);
  A.census = d;
  rc = td_launch_pair(s->dp, A, s->pair_nt, s->pair_split, s->nl_skin > 0.0f, s->sA);
  s->launches += 1;
  if (rc) { cudaFree(d); return fail(s, TDPD_ECUDA, "pair kernel attribute"); }
  CK(cudaMemcpyAsync(n_front, d, n * 4, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaMemcpyAsync(xor_front, d + n, n * 4, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaMemcpyAsync(n_ring, d + 2 * n, n * 4, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaMemcpyAsync(xor_ring, d + 3 * n, n * 4, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaStreamSynchronize(s->sA));
  cudaFree(d);
  s->have_forces = false;  // F4 / Qx were not written by this launch: re-evaluate before they are used again
  return TDPD_OK;
}

extern "C" int tdpd_debug_set_run_meta(tdpd_sim* s, uint32_t run_index, uint32_t meta) {
  if (!s || !s->finalized || run_index >= s->seg_meta.size()) return TDPD_EINVAL;
  int rc = tdpd_sync(s);
  if (rc) return rc;
  CK(cudaMemcpy(s->seg_meta_d + run_index, &meta, 4, cudaMemcpyHostToDevice));
  s->have_forces = false;
  drop_graphs(s);
  return TDPD_OK;
}

extern "C" int tdpd_debug_rng(tdpd_sim* s, int64_t n, const int64_t* id_i, const int64_t* id_j, int64_t step,
                              uint32_t tag, uint32_t* words, float* gauss) {
  if (!s || n < 0 || !id_i || !id_j) return TDPD_EINVAL;
  if (n == 0) return TDPD_OK;
  CK(cudaSetDevice(s->device));
  int64_t *di = nullptr, *dj = nullptr;
  uint32_t* dw = nullptr;
  float* dg = nullptr;
  CK(cudaMalloc(&di, n * 8)); CK(cudaMalloc(&dj, n * 8)); CK(cudaMalloc(&dw, n * 16)); CK(cudaMalloc(&dg, n * 16));
  CK(cudaMemcpyAsync(di, id_i, n * 8, cudaMemcpyHostToDevice, s->sA));
  CK(cudaMemcpyAsync(dj, id_j, n * 8, cudaMemcpyHostToDevice, s->sA));
  td_launch_rng_debug(s->dp, n, di, dj, (uint32_t)step, tag, dw, dg, s->sA);
  s->launches += 1;
  if (words) CK(cudaMemcpyAsync(words, dw, n * 16, cudaMemcpyDeviceToHost, s->sA));
  if (gauss) CK(cudaMemcpyAsync(gauss, dg, n * 16, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaStreamSynchronize(s->sA));
  cudaFree(di); cudaFree(dj); cudaFree(dw); cudaFree(dg);
  return TDPD_OK;
}

extern "C" int tdpd_debug_box_muller(tdpd_sim* s, int64_t n, const uint32_t* words, float* gauss) {
  if (!s || n < 0 || !words || !gauss) return TDPD_EINVAL;
  if (n == 0) return TDPD_OK;
  CK(cudaSetDevice(s->device));
  uint32_t* dw = nullptr;
  float* dg = nullptr;
  CK(cudaMalloc(&dw, n * 8)); CK(cudaMalloc(&dg, n * 8));
  CK(cudaMemcpyAsync(dw, words, n * 8, cudaMemcpyHostToDevice, s->sA));
  td_launch_box_muller_debug(n, dw, dg, s->sA);
  s->launches += 1;
  CK(cudaMemcpyAsync(gauss, dg, n * 8, cudaMemcpyDeviceToHost, s->sA));
  CK(cudaStreamSynchronize(s->sA));
  cudaFree(dw); cudaFree(dg);
  return TDPD_OK;
}

extern "C" int tdpd_host_grid(const tdpd_params* p, int32_t ncell[3], uint32_t* n_runs, uint32_t* cell_rank,
                              uint32_t* seg_off, uint32_t* seg_first, uint32_t* seg_meta) {
  std::string why;
  if (!validate_params(p, why)) return TDPD_EINVAL;
  tdpd_sim tmp;  // host-only: no CUDA call is made
  tmp.prm = *p;
  derive_params(*p, tmp.dp);
  build_grid(&tmp);
  if (ncell) for (int a = 0; a < 3; ++a) ncell[a] = tmp.dp.ncell[a];
  if (n_runs) *n_runs = (uint32_t)tmp.seg_first.size();
  if (cell_rank) memcpy(cell_rank, tmp.cell_rank.data(), tmp.cell_rank.size() * 4);
  if (seg_off) memcpy(seg_off, tmp.seg_off.data(), tmp.seg_off.size() * 4);
  if (seg_first) memcpy(seg_first, tmp.seg_first.data(), tmp.seg_first.size() * 4);
  if (seg_meta) memcpy(seg_meta, tmp.seg_meta.data(), tmp.seg_meta.size() * 4);
  return TDPD_OK;
}

extern "C" int tdpd_set_timing(tdpd_sim* s, int32_t on) {
  if (!s) return TDPD_EINVAL;
  tdpd_sync(s);
  for (auto& t : s->timers) {
    for (auto& e : t.ev) { cudaEventDestroy(e.first); cudaEventDestroy(e.second); }
    t.ev.clear(); t.launches = 0; t.ms = 0;
  }
  s->timing = on != 0;
  return TDPD_OK;
}

extern "C" int tdpd_get_timing(tdpd_sim* s, int64_t launches[TDPD_N_TIMERS], double ms[TDPD_N_TIMERS]) {
  if (!s) return TDPD_EINVAL;
  int rc = tdpd_sync(s);
  if (rc) return rc;
  for (int k = 0; k < TDPD_N_TIMERS; ++k) {
    Timer& t = s->timers[k];
    for (auto& e : t.ev) {
      float m = 0.f;
      if (cudaEventElapsedTime(&m, e.first, e.second) == cudaSuccess) t.ms += m;
      cudaEventDestroy(e.first); cudaEventDestroy(e.second);
    }
    t.ev.clear();
    if (launches) launches[k] = t.launches;
    if (ms) ms[k] = t.ms;
  }
  return TDPD_OK;
}

extern "C" int64_t tdpd_launch_count(const tdpd_sim* s) { return s ? s->launches : 0; }

extern "C" int tdpd_set_tuning(tdpd_sim* s, int32_t pair_threads, int32_t list_cap, int32_t pair_split) {
  if (!s) return TDPD_EINVAL;
  if (s->finalized) return fail(s, TDPD_ESTATE, "tuning must be set before tdpd_set_workspace");
  if (pair_threads != 0 && pair_threads != 32 && pair_threads != 64 && pair_threads != 128 && pair_threads != 256)
    return fail(s, TDPD_EINVAL, "pair_threads must be 0, 32, 64, 128 or 256");
  if (list_cap != 0 && (list_cap < 4 || list_cap > 400)) return fail(s, TDPD_EINVAL, "list_cap must be 0 or 4..400");
  if (pair_split != 0 && pair_split != 1 && pair_split != 2 && pair_split != 4 && pair_split != 16)
    return fail(s, TDPD_EINVAL, "pair_split must be 0, 1, 2, 4 or 16");
  s->tune_nt = pair_threads;
  s->tune_split = pair_split;
  s->tune_lcap = list_cap;
  return TDPD_OK;
}

extern "C" int tdpd_set_neighbor_list(tdpd_sim* s, float skin, int32_t list_cap) {
  if (!s) return TDPD_EINVAL;
  if (s->finalized) return fail(s, TDPD_ESTATE, "the neighbour-list mode must be chosen before tdpd_set_workspace");
  if (!(skin >= 0.0f) || list_cap < 0 || list_cap > 4096) return fail(s, TDPD_EINVAL, "skin >= 0 and 0 <= list_cap <= 4096");
  if (skin > 0.0f) {
    double rl = (double)std::max(s->prm.r_c, s->prm.r_cc) + (double)skin;
    for (int a = 0; a < 3; ++a)
      if ((int)std::floor((double)s->prm.box[a] / rl) < 3)
        return fail(s, TDPD_EINVAL, "box smaller than 3 cells of edge cutoff + skin per axis");
  }
  s->nl_skin = skin;
  s->tune_nl_cap = list_cap;
  derive_params(s->prm, s->dp, skin);
  s->seg_off.clear();  // the grid changed: rebuild the static neighbour runs
  return TDPD_OK;
}

extern "C" int tdpd_get_neighbor_list_stats(tdpd_sim* s, int64_t* n_rebuilds, int64_t* n_evaluations, int32_t* list_cap,
                                            int32_t* max_entries) {
  if (!s) return TDPD_EINVAL;
  if (n_rebuilds) *n_rebuilds = 0;
  if (n_evaluations) *n_evaluations = 0;
  if (list_cap) *list_cap = s->nl_cap;
  if (max_entries) *max_entries = 0;
  if (!(s->nl_skin > 0.0f) || !s->finalized) return TDPD_OK;
  int rc = tdpd_sync(s);
  if (rc) return rc;
  uint32_t w[8];
  CK(cudaMemcpy(w, s->step_d, sizeof w, cudaMemcpyDeviceToHost));
  if (n_rebuilds) *n_rebuilds = w[TD_CTL_NREBUILD];
  if (n_evaluations) *n_evaluations = w[TD_CTL_NDECIDE];
  if (max_entries && s->n) {
    std::vector<uint32_t> c((size_t)s->n);
    CK(cudaMemcpy(c.data(), s->nl_cnt_d, (size_t)s->n * 4, cudaMemcpyDeviceToHost));
    *max_entries = (int32_t)*std::max_element(c.begin(), c.end());
  }
  return TDPD_OK;
}

extern "C" int tdpd_set_membrane_variant(tdpd_sim* s, int32_t previous_step_area_volume) {
  if (!s) return TDPD_EINVAL;
  s->lag_av = previous_step_area_volume != 0;
  s->have_forces = false;
  drop_graphs(s);  // the flag is a kernel argument of the captured nodes
  return TDPD_OK;
}

extern "C" int tdpd_set_graph(tdpd_sim* s, int32_t on) {
  if (!s) return TDPD_EINVAL;
  s->use_graph = on != 0;
  if (!on) drop_graphs(s);
  return TDPD_OK;
}

extern "C" const char* tdpd_last_error(const tdpd_sim* s) { return s ? s->err.c_str() : "null handle"; }

extern "C" int tdpd_destroy(tdpd_sim* s) {
  if (!s) return TDPD_EINVAL;
  cudaSetDevice(s->device);
  cudaStreamSynchronize(s->sA);
  cudaStreamSynchronize(s->sB);
  for (auto& t : s->timers)
    for (auto& e : t.ev) { cudaEventDestroy(e.first); cudaEventDestroy(e.second); }
  drop_graphs(s);
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  if (s->ev_join) cudaEventDestroy(s->ev_join);
  if (s->own_streams) { cudaStreamDestroy(s->sA); cudaStreamDestroy(s->sB); }
  if (s->own_ws && s->ws) cudaFree(s->ws);
  delete s;
  return TDPD_OK;
}
