/*
 * tdpd.h — C ABI of libtdpd.so: the per-timestep hot path of transport Dissipative Particle Dynamics
 * (tDPD) with explicit red-blood-cell membranes (arXiv:1611.06163) on ONE NVIDIA B200 (sm_100a).
 *
 * Citations are /root/reference/PAPER.md:<line> (+ equation) and DESIGN.md readings R<n>.
 *
 * The path behind tdpd_step (every stage is a hand-written CUDA kernel; there is no CPU fallback):
 *   a1-a3  cell-list binning: wrap + cell hash in Morton order, stable radix sort, cell-start table, reorder
 *
 *   a4     non-bonded pair kernel: F_i = sum_j [F^C + F^D + F^R] (Eq 2-6) for r < r_c and
 *          Q_i = sum_j [Q^D + Q^R] (Eq 7-10) for r < r_cc, both sides of each pair, no atomics
 *   a5-a8  membrane kernel: WLC+POW bonds with dissipative/random terms (Eq 13-16), K-Gather of
 *          total area/volume and K-Apply of the area/volume constraints (Eq 17-18),
 *          dihedral bending (Eq 19)
 *   a9     fused velocity-Verlet of position, velocity and concentration (R21; the paper is silent)
 *   a10    a4 and a5-a8 run on two caller-supplied CUDA streams joined by events
 *
 * Conventions
 *   - Up to TDPD_MAX_SPECIES = 10 chemical species, concentrations [n][n_species] species-fastest.
 *   - All array arguments are HOST pointers, caller-owned, C-contiguous; the library copies in / out.
 *     The only DEVICE pointer is the workspace given to tdpd_set_workspace (caller-owned device memory, e.g. a
 *     torch uint8 tensor); the library owns its contents until tdpd_destroy.
 *   - Particle ids are persistent: 0..n-1 in the order of the load/add calls.  Every get_* returns arrays in
 *     id order regardless of the internal (cell-sorted) order.
 *   - Every function returns TDPD_OK (0) or a negative error code; tdpd_last_error gives a message.
 *     Nothing throws, aborts or prints across this boundary.
 *   - One handle is used from one host thread at a time.
 *   - Random numbers: Philox-4x32-10, counter = (min id, max id, step word k, tag), key = seed (DESIGN.md R-RNG).
 *     Force evaluation number k uses step word k; the evaluation at load time is k = 0; after tdpd_step(n) the
 *     step counter is n.  Results do not depend on how steps are batched.
 */
#ifndef TDPD_H
#define TDPD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TDPD_MAX_TYPES 4
#define TDPD_MAX_SPECIES 10 /* the paper benchmarks up to N_spec = 10 */

enum {
  TDPD_OK = 0,
  TDPD_EINVAL = -1,    /* bad argument, box smaller than 3 cells per axis, type out of range, open mesh ... */
  TDPD_ESTATE = -2,    /* call order: step before workspace, load after workspace, ... */
  TDPD_ENOMEM = -3,    /* workspace too small / allocation failed */
  TDPD_ECUDA = -4,     /* a CUDA call failed; see tdpd_last_error */
  TDPD_EUNSTABLE = -5  /* NaN / Inf in the state, or a WLC bond reached x >= 1, seen at tdpd_get_state */
};

enum { TDPD_BODY_OFF = 0, TDPD_BODY_UNIFORM = 1, TDPD_BODY_DOUBLE_POISEUILLE_Z = 2 };

/* Model and run parameters (POD).  struct_size must be sizeof(tdpd_params). */
typedef struct tdpd_params {
  uint32_t struct_size;
  int32_t n_types;    /* 1..TDPD_MAX_TYPES   */
  int32_t n_species;  /* 1..TDPD_MAX_SPECIES */
  float box[3];       /* periodic box lengths; >= 3 cells of edge max(r_c, r_cc) per axis */
  float r_c;          /* force cutoff (Eq 3-5) */
  float r_cc;         /* flux cutoff (Eq 8-9)  */
  float dt;
  float kBT;
  float rho;          /* number density entering Eq 10 (R6) */
  float a[TDPD_MAX_TYPES][TDPD_MAX_TYPES];      /* Eq 3 alpha_ij; must be symmetric */
  float gamma[TDPD_MAX_TYPES][TDPD_MAX_TYPES];  /* Eq 4 gamma_ij; sigma_ij^2 = 2 kBT gamma_ij (Eq 6) */
  float s_R[TDPD_MAX_TYPES][TDPD_MAX_TYPES];    /* omega_R = (1 - r/r_c)^s_R, omega_D = omega_R^2 (R3) */
  float kappa[TDPD_MAX_SPECIES][TDPD_MAX_TYPES][TDPD_MAX_TYPES]; /* Eq 8 kappa_ij per species (R15) */
  float s_c[TDPD_MAX_SPECIES];                  /* omega_DC = (1 - r/r_cc)^s_c (R4) */
  float m_s[TDPD_MAX_SPECIES];                  /* Eq 10 m_s; 0 switches the random flux off */
  float body_force[3];
  int32_t body_mode;  /* TDPD_BODY_* (R14) */
  uint64_t seed;
  int32_t exclude_same_cell_membrane_pairs;     /* R16 */
  int32_t reserved;
  /* Source term of Eq 7 (PAPER.md:63, :78 "external concentration source", :272 "reacts with the solvent and
   * dissipates"; the paper gives no form: DESIGN.md reading R-QS): Q^S_i = source[s][type_i] - decay[s][type_i] C_i^s,
   * added to the flux of every force evaluation.  All zero = no source. */
  float source[TDPD_MAX_SPECIES][TDPD_MAX_TYPES];
  float decay[TDPD_MAX_SPECIES][TDPD_MAX_TYPES];
} tdpd_params;

/* Membrane model parameters (values are inputs, R11). */
typedef struct tdpd_rbc_params {
  float p;        /* WLC persistence length (Eq 13) */
  float x0;       /* h_m / h_0 */
  float m;        /* POW exponent (Eq 14) */
  float gamma_T, gamma_C;   /* Eq 15; requires 3 gamma_C >= gamma_T (Eq 16) */
  float k_g, k_l, k_v;      /* Eq 17-18 */
  float k_b, theta0;        /* Eq 19 */
  float VR_over_AR32;       /* V^R / (A^R)^{3/2} */
} tdpd_rbc_params;

typedef struct tdpd_sim tdpd_sim; /* opaque, library-owned */

/* Creates an empty simulation on CUDA device `device`.  stream_pair / stream_bonded are caller-owned
 * cudaStream_t handles (e.g. torch.cuda.Stream().cuda_stream); NULL selects library-created streams.
 * EINVAL: bad struct_size / ranges / asymmetric tables / box too small. */
int tdpd_create(const tdpd_params* p, int device, void* stream_pair, void* stream_bonded, tdpd_sim** out);

/* Appends n free particles (position, velocity, concentration of every species).
 * pos [n][3] inside [0, box) (values outside are wrapped once), vel [n][3] or NULL (zero), type [n] or NULL
 * (type 0), conc [n][n_species] or NULL (zero).  ESTATE after tdpd_set_workspace. */
int tdpd_load_particles(tdpd_sim* s, int64_t n, const float* pos, const float* vel, const int32_t* type,
                        const float* conc);

/* Appends one closed triangulated membrane: nv vertices (box coordinates, may straddle the
 * periodic boundary), ntri triangles tri[ntri][3] of local vertex indices, counter-clockwise seen from outside.
 * The library derives the bonds (unique edges), one dihedral per shared edge, per-bond rest length h_0 = initial
 * length and k_p from force balance at h_0 (R11), per-triangle A_0t, A_0 = sum A_0t and
 * V_0 = A_0^{3/2} V^R/(A^R)^{3/2}.  Vertices get particle type `mtype`.
 * *rbc_index_out (may be NULL) receives the 0-based membrane index.
 * EINVAL: mesh not a closed consistently oriented manifold, nv > 65535, 3 gamma_C < gamma_T. */
int tdpd_add_rbc_mesh(tdpd_sim* s, int32_t nv, const float* verts, const float* vel, const float* conc,
                      int32_t ntri, const int32_t* tri, const tdpd_rbc_params* rp, int32_t mtype,
                      int32_t* rbc_index_out);

/* Device bytes needed for everything loaded so far. */
int tdpd_workspace_bytes(const tdpd_sim* s, size_t* bytes);

/* Hands the library its device memory (256-byte aligned, >= tdpd_workspace_bytes) and uploads the system.
 * dev_ptr == NULL: the library allocates with cudaMalloc and frees at destroy.  After this call the particle
 * set is frozen.  ENOMEM: too small. */
int tdpd_set_workspace(tdpd_sim* s, void* dev_ptr, size_t bytes);

/* Replaces the parameters; takes effect at the next force evaluation (the current forces are re-evaluated with
 * the current step word before the next step).  The cell grid and the type/species counts must not change
 * after tdpd_set_workspace, and kBT, dt and the box must not change once a membrane is loaded (its k_p, h_0, A_0,
 * V_0 were derived from them at tdpd_add_rbc_mesh): EINVAL. */
int tdpd_set_params(tdpd_sim* s, const tdpd_params* p);

/* Overwrites positions / velocities / concentrations of all particles in id order (any pointer may be NULL),
 * keeps the step counter.  Forces are re-evaluated with the current step word.  Returns after the host buffers
 * have been copied: the caller may reuse them at once. */
int tdpd_set_state(tdpd_sim* s, const float* pos, const float* vel, const float* conc);

/* Advances nsteps velocity-Verlet steps (R21).  Asynchronous: only enqueues work on the two streams. */
int tdpd_step(tdpd_sim* s, int32_t nsteps);

/* Blocks until all enqueued work is done. */
int tdpd_sync(tdpd_sim* s);

/* Copies out, in id order: pos [n][3], vel [n][3], conc [n][S], force [n][3] (pair + bonded, without the body
 * term), flux [n][S], *step.  Any pointer may be NULL.  All requested arrays are gathered and copied asynchronously,
 * then the call synchronises once.  EUNSTABLE if a value is not finite, a bond is overstretched or a list overflowed. */
int tdpd_get_state(tdpd_sim* s, float* pos, float* vel, float* conc, float* force, float* flux, int64_t* step);

/* Same as the force part of tdpd_get_state, split into the non-bonded and the membrane contribution. */
int tdpd_get_forces_split(tdpd_sim* s, float* force_pair, float* force_bonded);

int64_t tdpd_num_particles(const tdpd_sim* s);
int32_t tdpd_num_rbc(const tdpd_sim* s);

/* Per membrane: total area and volume of the last force evaluation (K-Gather) and the targets.
 * Any pointer may be NULL.  Synchronises. */
int tdpd_get_rbc_stats(tdpd_sim* s, double* area, double* volume, double* A0, double* V0);

/* Derived topology of membrane m (for tests): nbond, then bond[nbond][2], dih[nbond][4], h0, kp (per bond),
 * A0t (per triangle); any array may be NULL. */
int tdpd_get_rbc_topology(tdpd_sim* s, int32_t m, int32_t* nbond, int32_t* bond, int32_t* dih, float* h0,
                          float* kp, float* A0t);

/* Binning of the current positions (bit-exact test, DESIGN.md R-bin): cell_xyz [n][3] by id,
 * ncell[3], cell_count [ncell_x*ncell_y*ncell_z] x-fastest (may be NULL), and sorted_id [n]: the id held by each
 * slot of the cell-sorted order (may be NULL). */
int tdpd_debug_get_binning(tdpd_sim* s, int32_t* cell_xyz, int32_t ncell[3], int32_t* cell_count,
                           int32_t* sorted_id);

/* Neighbour census through the cell list of the current positions (exact arithmetic on the fp32 positions):
 * per id the number of neighbours within r_c and r_cc and the XOR of their ids (same-membrane pairs and
 * coincident particles excluded exactly as in the force sum). */
int tdpd_debug_neighbor_census(tdpd_sim* s, int32_t* n_rc, int32_t* n_rcc, uint32_t* xor_rc, uint32_t* xor_rcc);

/* The hit lists of the pair kernel itself (bit-exact indexing test): runs the REAL pair kernel (same neighbour-run
 * tables, candidate loops, thresholds and hit stacks as a force evaluation, in the launch configuration in use) with
 * the evaluation replaced by a count: per id the number of entries on the front list (r < min(r_c, r_cc)) and on
 * the ring list (up to max(r_c, r_cc)) and the XOR of the ids behind them; same-membrane and coincident pairs are
 * left out as in the force sum.  The list thresholds are the cutoffs inflated by 1e-6 relative (DESIGN.md R-cut), so
 * a pair within that band of a cutoff may sit on either side. */
int tdpd_debug_pair_census(tdpd_sim* s, int32_t* n_front, int32_t* n_ring, uint32_t* xor_front, uint32_t* xor_ring);

/* Test support: overwrites word `run_index` of the device copy of the static neighbour-run table (seg_meta of
 * tdpd_host_grid), so that a test can show the indexing checks notice a wrong table entry. */
int tdpd_debug_set_run_meta(tdpd_sim* s, uint32_t run_index, uint32_t meta);

/* Raw random stream of the device path (for the bit-exact Philox test and the Gaussian tolerance test):
 * words [n][4] = Philox-4x32-10 of counter (min(id_i,id_j), max(id_i,id_j), step, tag) with the simulation's
 * seed; gauss [n][4] = the four Gaussians the kernels derive from them (fp32).  Either may be NULL. */
int tdpd_debug_rng(tdpd_sim* s, int64_t n, const int64_t* id_i, const int64_t* id_j, int64_t step, uint32_t tag,
                   uint32_t* words, float* gauss);

/* Box-Muller of caller-chosen raw words through the device functions the kernels use: words [n][2] = (x_a, x_b),
 * gauss [n][2] = R(x_a) (cos 2 pi u(x_b), sin 2 pi u(x_b)).  Lets a test reach the u -> 1 branch of the radius. */
int tdpd_debug_box_muller(tdpd_sim* s, int64_t n, const uint32_t* words, float* gauss);

/* Host-only view of the static grid tables the pair kernel uses (no CUDA device needed; for tests): ncell[3] per
 * R-bin, cell_rank [ncells] (x-fastest linear cell -> Morton rank), and the neighbour runs of every cell in CSR form
 * by Morton rank: seg_off [ncells + 1], seg_first [*n_runs] (first Morton rank of the run), seg_meta [*n_runs]
 * (cells in the run | (wrap_x + 1) << 4 | (wrap_y + 1) << 6 | (wrap_z + 1) << 8).  Call once with NULL arrays to get
 * ncell and *n_runs.  A run is a set of rank-consecutive neighbour cells of one 2x2x2 block and one periodic image. */
int tdpd_host_grid(const tdpd_params* p, int32_t ncell[3], uint32_t* n_runs, uint32_t* cell_rank, uint32_t* seg_off,
                   uint32_t* seg_first, uint32_t* seg_meta);

/* Per-kernel timing with CUDA events on the launching streams (bench.py's roofline leg).  While enabled every
 * launch of the kernels below is bracketed by an event pair; tdpd_get_timing synchronises and returns, per
 * kernel class, the number of launches and the summed milliseconds since tdpd_set_timing(s, 1).
 * Classes: 0 integrate (kick/drift/key), 1 sort, 2 reorder + cell table, 3 pair, 4 membrane, 5 closing kick,
 * 6 neighbour list (rebuild decision + list build; neighbour-list mode only). */
#define TDPD_N_TIMERS 7
int tdpd_set_timing(tdpd_sim* s, int32_t on);
int tdpd_get_timing(tdpd_sim* s, int64_t launches[TDPD_N_TIMERS], double ms[TDPD_N_TIMERS]);

/* Measured denominators of the pair kernel's roofline, taken by microbenchmarks on `device` (about
 * 0.3 s, not on the timed path): FP32 FMA throughput with scalar fma (three register operands) and with the packed
 * fma.rn.f32x2 of sm_100 (FFMA2), read bandwidth of a 32 MB L2-resident buffer and of a 1 GiB buffer (HBM), the SM
 * count.  ECUDA / ENOMEM on failure. */
typedef struct tdpd_peaks {
  double fp32_fma_tflops, fp32_fma2_tflops, l2_read_gbs, hbm_read_gbs;
  int32_t n_sm, reserved;
} tdpd_peaks;
int tdpd_measure_peaks(int device, tdpd_peaks* out);

/* Number of kernels the library launched since creation (bench.py's gpu_launches). */
int64_t tdpd_launch_count(const tdpd_sim* s);

/* Pair-kernel launch knobs (tuning; results are identical up to the fp32 summation order of a particle's
 * neighbours): pair_threads in {32, 64, 128, 256} = threads per CTA, list_cap in 4..400 = entries of the
 * per-thread neighbour list in shared memory (a full list is evaluated early, never overflowed), pair_split in
 * {1, 2, 4, 16} = threads per particle (sub-wave systems); 0 = automatic.  ESTATE after tdpd_set_workspace. */
int tdpd_set_tuning(tdpd_sim* s, int32_t pair_threads, int32_t list_cap, int32_t pair_split);

/* the paper's own operating regime ("Neighbor lists were updated every 5 steps";
 * construction and transposed layout PAPER.md:136-138).  skin > 0 switches the neighbour-list mode on: the cells get
 * an edge >= max(r_c, r_cc) + skin, every binning also writes, per particle, the list of all particles within
 * cutoff + skin (16-bit entries, [tile of 256 slots][entry][lane]), and the following steps skip sort, reorder and
 * the 27-cell scan: the pair kernel re-tests the list entries against the true cutoffs with the current positions.
 * After the drift of every step the device takes the largest displacement d_max since the last binning and re-bins
 * in that same step iff 2 d_max > skin (a pair inside a cutoff could otherwise be missing), so the forces are those of
 * the every-step binning up to the fp32 summation order.  list_cap = entries per particle (0: 1.5 x the mean + 32);
 * a fuller neighbourhood sets an error reported by tdpd_get_state (EUNSTABLE).  skin = 0 switches the mode off.
 * ESTATE after tdpd_set_workspace; EINVAL if the box has fewer than 3 cells of edge cutoff + skin per axis. */
int tdpd_set_neighbor_list(tdpd_sim* s, float skin, int32_t list_cap);

/* Neighbour-list mode: binnings (list rebuilds) and force evaluations since creation, the list capacity and the
 * longest list of the last binning.  Any pointer may be NULL.  Synchronises. */
int tdpd_get_neighbor_list_stats(tdpd_sim* s, int64_t* n_rebuilds, int64_t* n_evaluations, int32_t* list_cap,
                                 int32_t* max_entries);

/* SURVEY §8(f) row 3 (Fig 2): 1 = K-Apply takes the total area and volume of the force evaluation of the
 * PREVIOUS time step instead of this step's (the very first evaluation and one that follows tdpd_set_state use their
 * own), so that the constraint forces do not wait for this launch's reduction; 0 (default) = sequential variant, the
 * definition (R20).  May be called at any time; the forces are re-evaluated. */
int tdpd_set_membrane_variant(tdpd_sim* s, int32_t previous_step_area_volume);

/* Steps are replayed as CUDA graphs (one per ping-pong side x first/last step of a call, captured on first use) unless
 * per-kernel timing is on; on = 0 switches to plain launches.  Results are bit-identical either way. */
int tdpd_set_graph(tdpd_sim* s, int32_t on);

/* ---- Sorting without allocating ------------------------------------------------------------------------------------
 * The stable LSD radix sort of (cell key, previous slot) pairs of row a2 (PAPER.md:137 "particle reordering", :141
 * "radix sort"), the same kernels a step runs, as a call of its own for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, tight serving loops): its scratch (digit histograms, chunk totals and the
 * second side of the ping-pong) is one fixed device array inside the library, TDPD_NOALLOC_SCRATCH_BYTES on every GPU
 * that loads the library until the process exits.  The call allocates nothing and frees nothing.
 *   d_keys      [n] DEVICE, read only: 32-bit keys, only the low key_bits bits (1..32) are significant
 *   d_vals      [n] DEVICE, read only, or NULL for the values 0 .. n-1 (the result is then the sorting permutation)
 *   d_keys_out  [n] DEVICE: the keys in ascending order; equal keys keep their input order (stable)
 *   d_vals_out  [n] DEVICE: the values in the order of their keys
 *   stream      a cudaStream_t (NULL = the default stream); the call only enqueues work and does not synchronise
 * d_keys_out may be d_keys and d_vals_out may be d_vals (in place); any other overlap of the four arrays is not allowed.
 * The pointers must belong to the CURRENT device of the calling thread.  The caller keeps ownership of all four.
 * n <= TDPD_NOALLOC_MAX_N, else TDPD_EINVAL (nothing is enqueued); other bad arguments TDPD_EINVAL, CUDA errors
 * TDPD_ECUDA; the message of the calling thread's last failure is tdpd_noalloc_last_error.  n = 0 is a no-op.
 * All calls on a device share the one scratch array, which keeps the contents of the last call (nothing in it has to
 * start at zero: every entry a call reads was written by that call).  Calls whose kernels can overlap on the GPU
 * (different streams without an event between them, several host threads) RACE: keep them on one stream.
 * tdpd_noalloc_init asks the driver for the array's address on the current device (done once per device, otherwise
 * on the first sort there): call it before a stream capture begins. */
#define TDPD_NOALLOC_MAX_N 262144
#define TDPD_NOALLOC_SCRATCH_BYTES 2228224 /* 2 x 4 x MAX_N of ping-pong + 128 KiB of histograms */
int tdpd_noalloc_init(void);
int tdpd_sort_cells_noalloc(const uint32_t* d_keys, const uint32_t* d_vals, int64_t n, int32_t key_bits,
                            uint32_t* d_keys_out, uint32_t* d_vals_out, void* stream);
const char* tdpd_noalloc_last_error(void);

const char* tdpd_last_error(const tdpd_sim* s);
int tdpd_destroy(tdpd_sim* s);

#ifdef __cplusplus
}
#endif
#endif /* TDPD_H */
