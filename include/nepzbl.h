/*
 * nepzbl.h -- C ABI of the B200-native NEP-ZBL hot path (arXiv 2305.08140).
 *
 * One library, libnepzbl.so, built from paper_2305_08140_b200/csrc for sm_100a.  Every step of the
 * path -- state prep, cell-list neighbour build, radial/angular descriptors, network, force/virial
 * back-pass, ZBL pair term, velocity-Verlet with adaptive time step -- runs in its CUDA kernels.
 * There is no CPU fallback: without a CUDA device nep_zbl_create fails with NEPZBL_E_CUDA.
 *
 * Citations: P:n = PAPER.md line n; S:x = SURVEY.md section 8(c) paragraph x; D:x = DESIGN.md.
 *
 * Conventions
 *   - Units: eV, Angstrom, amu, fs.  1 amu*A^2/fs^2 = 103.6426965 eV.
 *   - "dev" pointers are device memory owned by the caller (e.g. torch tensors); "host" pointers
 *     are host memory owned by the caller.  The library never frees caller memory and the caller
 *     never frees library memory (the handle is released by nep_zbl_destroy only).
 *   - Positions / velocities are fp64 SoA: x[n] y[n] z[n] (3n doubles).  Forces are fp32 SoA [3n],
 *     virials fp32 SoA [9n] with component c = 3*alpha+beta at virial[c*n + i], energies fp64 [n].
 *     All per-atom results are in the CALLER's atom order (the library sorts internally).
 *   - box[9]: the three lattice vectors as ROW vectors, host.  pbc[3]: 1 periodic, 0 open (bulk periodic xyz;
 *     foil open in z).  Orthogonal boxes (off-diagonals == 0): any pbc; a periodic edge must be >= 2*(rc_radial+skin).
 *     Triclinic boxes (any off-diagonal != 0, C-28): periodic along all three lattice
 *     vectors (else NEPZBL_E_BOX_NOT_ORTHOGONAL); every distance between opposite cell faces must be
 *     >= 2*(rc_radial+skin); positions are wrapped along the lattice vectors.  The Wigner-Seitz count takes
 *     orthogonal boxes only.
 *   - All work is enqueued on the CUDA stream given at create.  Calls that return host scalars or
 *     status from the device (neighbor_build, nep_zbl_compute, md_step, md_run, md_energies,
 *     *_host) synchronise that stream before returning.
 *   - Every int-returning call returns NEPZBL_OK (0) or a negative NEPZBL_E_* code;
 *     nep_zbl_last_error gives a message.  Nothing is truncated silently: a neighbour list that
 *     does not fit cap_radial / cap_angular is an error that names the count needed.
 *   - Determinism: the same inputs give bit-identical outputs (no floating-point atomics; the only
 *     atomics are integer counters/max whose result does not depend on order).
 */
#ifndef NEPZBL_H
#define NEPZBL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nepzbl_handle nepzbl_handle; /* opaque, owned by the library */

enum {
  NEPZBL_OK = 0,
  NEPZBL_E_INVALID_ARG = -1,
  NEPZBL_E_BOX_NOT_ORTHOGONAL = -2, /* a non-orthogonal box with an open axis, or given to the Wigner-Seitz count */
  NEPZBL_E_BOX_TOO_SMALL = -3,     /* periodic edge < 2*(rc_radial+skin): minimum image invalid */
  NEPZBL_E_NEIGHBOR_OVERFLOW = -4, /* an atom has more neighbours than cap_radial / cap_angular */
  NEPZBL_E_NONFINITE = -5,         /* NaN/Inf in positions */
  NEPZBL_E_CUDA = -6,
  NEPZBL_E_UNSUPPORTED = -7,       /* model shape outside what this build instantiates */
  NEPZBL_E_WORKSPACE = -8,         /* workspace missing or too small */
  NEPZBL_E_STATE = -9              /* call order (e.g. md_step before md_init) */
};

/*
 * Model and list parameters.  Host memory; copied at create; the caller keeps ownership.
 * NEP-ZBL site energy (Eq. 1): U_i = U_i^NEP({q}) + 1/2 sum_j U_ZBL(r_ij).
 * Hyper-parameters as listed in P:106; functional forms per S:B-S:D (the paper defers them to its
 * ref. [25]).  Descriptor order (S:C): radial n = 0..n_max_radial; 3-body l-major
 * (l = 1..l_max, n = 0..n_max_angular); then the (2,2,2) 4-body term n = 0..n_max_angular; then the (1,1,1,1)
 * 5-body term n = 0..n_max_angular.
 */
typedef struct {
  int32_t n_types;                     /* 1 or 2 in this build */
  double rc_radial, rc_angular;        /* cutoffs r_c^R, r_c^A (6.0, 4.0 A) */
  int32_t n_max_radial, n_max_angular; /* n = 0..n_max; <= 15 / 10 (<= 4 / 4 with the 5-body term, or the 4-body term and two types) */
  int32_t basis_radial, basis_angular; /* Chebyshev basis k = 0..basis (D: C-2); <= 8.  A model smaller than the kernel
                                          shape it runs on is zero-padded to it at create; other sizes: NEPZBL_E_UNSUPPORTED */
  int32_t l_max;                       /* Legendre order of the 3-body part (4) */
  int32_t has_4body;                   /* 1: (l1,l2,l3) = (2,2,2) term */
  int32_t has_5body;                   /* 1: (l1,l2,l3,l4) = (1,1,1,1) term behind the 4-body block (D: C-27) */
  int32_t n_neurons;                   /* hidden tanh neurons */
  const double *c_radial;              /* [n_types][n_types][n_max_radial+1][basis_radial+1] */
  const double *c_angular;             /* [n_types][n_types][n_max_angular+1][basis_angular+1] */
  const double *q_scaler;              /* [D] (D: C-6) */
  const double *w0;                    /* [n_neurons][D] */
  const double *b0;                    /* [n_neurons] */
  const double *w1;                    /* [n_neurons] */
  double b1;
  int32_t zbl_enabled;                 /* Eq. 2 */
  double zbl_r_inner, zbl_r_outer;     /* Tersoff switch (1.0, 2.0 A) */
  int32_t zbl_n_terms;                 /* <= 4 */
  double zbl_c[4], zbl_d[4];           /* phi(x) = sum_k c_k exp(-d_k x)  (Eq. 3) */
  double zbl_a_num, zbl_a_pow;         /* a = a_num / (Z_i^pow + Z_j^pow)  (Eq. 4) */
  double coulomb_k;                    /* e^2/(4 pi eps0) in eV*A */
  const double *atomic_number;         /* [n_types] */
  const double *mass;                  /* [n_types], amu */
  double skin;                         /* neighbour-list skin, A (D: C-15) */
  int32_t cap_radial, cap_angular;     /* list capacities per atom (cap_radial <= 1024, cap_angular <= 128) */
} nepzbl_params;

/* Create a handle on CUDA device `device`; all work goes to `cuda_stream` (a cudaStream_t).  With NULL the library
 * creates its own BLOCKING stream: it is ordered against work on the legacy default stream exactly as the default
 * stream itself would be (so a caller that issues its own work there needs no extra synchronisation), but it can be
 * captured, so MD steps are still replayed as a CUDA graph.  Uploads the parameters (S1 of the path needs none).
 * Atom types must lie in [0, n_types); a type outside is reported as NEPZBL_E_INVALID_ARG by the call that reads it. */
int nep_zbl_create(const nepzbl_params *params, int device, void *cuda_stream, nepzbl_handle **out);
void nep_zbl_destroy(nepzbl_handle *h);
const char *nep_zbl_last_error(const nepzbl_handle *h); /* h may be NULL: create-time errors */
int nep_zbl_descriptor_dim(const nepzbl_handle *h);

/* Device workspace for up to n_atoms atoms.  The caller allocates it (e.g. a torch uint8 tensor),
 * hands it over with set_workspace and keeps it alive until destroy or the next set_workspace.
 * dev_ptr must be 256-byte aligned; n_atoms <= 2^28 = 268 435 456 per handle (the list build tags 28-bit atom
 * indices; about 3 KB of workspace per atom, so 180 GB hold ~55 million atoms anyway): NEPZBL_E_INVALID_ARG beyond. */
size_t nep_zbl_workspace_bytes(const nepzbl_handle *h, int64_t n_atoms);
int nep_zbl_set_workspace(nepzbl_handle *h, void *dev_ptr, size_t bytes, int64_t n_atoms);

/*
 * S2: cell-list neighbour build (BASELINE.json north_star; cutoffs P:106).  Sorts the atoms by
 * cell (canonical order), then lists for every atom all j with r_ij < rc_radial+skin (radial list)
 * and the subset r_ij < rc_angular+skin (angular list), minimum image on periodic axes, strict <.
 * pos_soa, types: dev.  box, pbc: host.
 */
int neighbor_build(nepzbl_handle *h, int64_t n, const double *pos_soa, const int32_t *types,
                   const double box[9], const int32_t pbc[3]);
/* Copy the current lists out, in the caller's atom indices: nn dev [n]; nl dev [n][cap] row-major
 * (entries beyond nn[i] are -1).  which: 0 radial, 1 angular.  Order inside a row is the
 * library's deterministic cell-walk order. */
int neighbor_get(nepzbl_handle *h, int which, int32_t *nn, int32_t *nl);

/*
 * S1,S3-S7: one NEP-ZBL evaluation (Eq. 1-4; S:B-S:E): per-atom energy, force, virial.
 * Reuses the current neighbour list when it is still valid for these positions (same n, box, pbc
 * and the two largest atomic displacements since the build add up to at most the skin), otherwise rebuilds it.
 * F_i = sum_j (dU_i/dr_ij - dU_j/dr_ji);  W_i = sum_j r_ij (x) dU_j/dr_ji  (r_ij = r_j - r_i), so
 * sum_i W_i = -dE/d(strain), positive under compression.  Any output pointer may be NULL.
 */
int nep_zbl_compute(nepzbl_handle *h, int64_t n, const double *pos_soa, const int32_t *types,
                    const double box[9], const int32_t pbc[3], double *energy, float *force,
                    float *virial);
/* Same call with HOST buffers: copies pos/types in and energy/force/virial out around the
 * evaluation (staging buffers live in the workspace). */
int nep_zbl_compute_host(nepzbl_handle *h, int64_t n, const double *pos_soa, const int32_t *types,
                         const double box[9], const int32_t pbc[3], double *energy, float *force,
                         float *virial);
/* Descriptor vectors of the last evaluation, fp32 dev [n][D] row-major, caller's atom order
 * (for parity tests of S3/S4). */
int nep_zbl_get_descriptors(nepzbl_handle *h, float *q);

/*
 * S8: velocity-Verlet with the adaptive time step of P:77 (S:F, D: C-11, C-12).
 * md_init registers caller-owned dev buffers pos_soa/vel_soa (integrated IN PLACE until destroy or
 * the next md_init), builds the list and evaluates the initial forces.
 * md_step: v_max = max_i |v_i|; dt = min(dt_max, max_displacement / v_max) (dt_max if v_max = 0);
 *   v += dt/2 F/m; x += dt v; wrap periodic axes; rebuild the list if the two largest displacements since
 *   the last build add up to more than the skin (C-15); F = F(x); v += dt/2 F/m.  Returns dt and
 *   whether the list was rebuilt (host).
 * md_run: n_steps such steps with no host round trip in between; dt_trace (host, [n_steps]) and
 *   n_rebuilds (host) may be NULL.
 * max_displacement may be +inf (fixed dt = dt_max).
 * A step is replayed as ONE CUDA graph (rebuild chain and ZBL kernel in device-set IF nodes).  ncu
 * cannot see kernels inside conditional graphs: the environment variable NEPZBL_NO_GRAPH=1, read
 * at nep_zbl_create, issues the same kernels as plain stream launches instead (same results).
 * NEPZBL_GATHER_BLOCK=32|64 (also read at create) fixes the threads per block of the two gather kernels, which
 * the library otherwise picks from the grid size (a tuning aid; results do not depend on it).
 * Other measurement switches read at create: NEPZBL_NN (network path, see nep_zbl_network_mode), NEPZBL_STAGE=1|2
 * (neighbour tiles of k_radial staged in shared memory by plain / bulk copies: measured slower, profiles/r2_staging.md),
 * NEPZBL_DENSE_THRESHOLD (fp64 re-evaluation thresholds, see nep_zbl_last_counts), NEPZBL_ANG_BLOCKS_PER_SM (size of the
 * angular kernel's persistent grid).  None changes what is computed beyond rounding.
 */
/* An MD session ends with destroy, the next md_init, nep_zbl_set_workspace -- or ANY neighbor_build /
 * nep_zbl_compute / nep_zbl_compute_host on the same handle (they overwrite the lists and the sorted order the session
 * and its captured graph rely on); md_step then returns NEPZBL_E_STATE until md_init is called again. */
int md_init(nepzbl_handle *h, int64_t n, double *pos_soa, double *vel_soa, const int32_t *types,
            const double box[9], const int32_t pbc[3]);
int md_step(nepzbl_handle *h, double dt_max, double max_displacement, double *dt_used,
            int32_t *rebuilt);
int md_run(nepzbl_handle *h, int64_t n_steps, double dt_max, double max_displacement,
           double *dt_trace, int64_t *n_rebuilds);
/* md_step with HOST state: copies pos/vel (host, 3n doubles each; pinned memory makes the copies
 * asynchronous) to the registered device buffers, steps, copies them back.  The new positions are final
 * after the drift, so their copy back runs on a second stream while the forces are evaluated; the call
 * returns when both buffers are complete. */
int md_step_host(nepzbl_handle *h, double *pos_soa, double *vel_soa, double dt_max,
                 double max_displacement, double *dt_used, int32_t *rebuilt);
/* The next md_step / first step of the next md_run rebuilds the neighbour list (S2) whatever the displacement
 * criterion says (asynchronous: one flag on the device).  bench.py uses it to put a list rebuild inside a short timed
 * region; a caller that edits positions by more than the skin between steps does not need it (the criterion sees the
 * edit). */
int md_request_rebuild(nepzbl_handle *h);
/* Total potential and kinetic energy of the current MD state (host scalars), fixed-order fp64
 * reduction. */
int md_energies(nepzbl_handle *h, double *e_pot, double *e_kin);
/* Current MD forces (fp32 SoA [3n]) and per-atom potential energies (fp64 [n]) to dev buffers. */
int md_get_forces(nepzbl_handle *h, float *force, double *energy);
/* Counters since md_init: steps, list rebuilds, ZBL pair evaluations of the last step. */
int md_get_counters(nepzbl_handle *h, int64_t *n_steps, int64_t *n_rebuilds, int64_t *n_zbl_atoms);

/*
 * Nose-Hoover chain thermostat on a group of atoms: "Atoms within a thickness of
 * 3 a0 of the boundaries of the simulation boxes ... are maintained at 300 K using the Nose-Hoover chain
 * thermostat [32]".  Equations of motion of ref. [32] with N_f = 3|G|, Q_1 = N_f k_B T tau^2,
 * Q_k = k_B T tau^2; every md_step / md_run step becomes NHC(dt/2) . velocity-Verlet(dt) . NHC(dt/2) with
 * dt still chosen from v(t) at the start of the step (C-24; the paper gives neither the chain
 * length, tau nor the splitting).
 * group: dev uint8 [n] in the caller's atom order, non-zero = thermostatted; caller-owned, must stay
 *   alive until destroy, the next md_init or md_set_thermostat(NULL, ...), which switches it off.
 * temperature in K, tau in fs, 1 <= chain_length <= 8.  Call after md_init; the chain starts at rest.
 * md_get_thermostat (host outputs, any may be NULL): chain positions xi[chain_length] and velocities
 *   vxi[chain_length] (1/fs), the group's kinetic temperature sum_G m v^2 / (N_f k_B) in K, and the
 *   thermostat's part of the conserved quantity of ref. [32],
 *   sum_k Q_k vxi_k^2 / 2 + N_f k_B T xi_1 + k_B T sum_{k>=2} xi_k  (eV).
 */
int md_set_thermostat(nepzbl_handle *h, const uint8_t *group, double temperature, double tau,
                      int32_t chain_length);
int md_get_thermostat(nepzbl_handle *h, double *xi, double *vxi, double *t_group, double *conserved_extra);
/* Restore the chain (host xi[chain_length], vxi[chain_length]) -- with the caller-owned pos / vel buffers this is
 * all a run needs to resume: md_init, md_set_thermostat, md_set_thermostat_state. */
int md_set_thermostat_state(nepzbl_handle *h, const double *xi, const double *vxi);

/*
 * Wigner-Seitz defect count: "The interstitials and vacancies were identified by
 * using the Wigner-Seitz cell methods [34]".  Every atom is assigned to the reference site nearest
 * to it (minimum image on periodic axes; exact for any atom position; ties go to the lowest site index,
 * DESIGN.md C-25); a site with no atom is a vacancy, a site with m >= 2 atoms holds m - 1 interstitials.
 * wigner_seitz_set_reference: site_soa dev fp64 [3][n_sites] (x[] y[] z[]), read during the call only
 *   (the library keeps its own cell-sorted copy, freed at destroy or at the next set_reference); box, pbc
 *   host.  Independent of the workspace and of md_init.
 * wigner_seitz_count: pos_soa dev fp64 [3][n] (any n; the atoms need not be the reference's).  Outputs:
 *   nearest dev int32 [n] (site index per atom, -1 for a non-finite position) or NULL; occupancy dev
 *   int32 [n_sites] or NULL; n_vacancies, n_interstitials host or NULL.  Synchronises the stream.
 */
int wigner_seitz_set_reference(nepzbl_handle *h, int64_t n_sites, const double *site_soa,
                               const double box[9], const int32_t pbc[3]);
int wigner_seitz_count(nepzbl_handle *h, int64_t n, const double *pos_soa, int32_t *nearest,
                       int32_t *occupancy, int64_t *n_vacancies, int64_t *n_interstitials);

/* 1 when md_step / md_run replay the step as a captured CUDA graph, 0 when they issue plain stream launches
 * (NEPZBL_NO_GRAPH=1, a failed capture -- nep_zbl_last_error then says why -- or no MD session). */
int nep_zbl_uses_graph(const nepzbl_handle *h);

/* Where the network layer (S6: descriptor x W0, tanh, dU/dq) of this handle runs:
 *   0  CUDA cores, FFMA with the weights broadcast from shared memory (k_angular_nn / k_angular_nn_split; every model;
 *      the only path for cap_angular > 64 and for neuron counts beyond the limits below)
 *   1  mma.sync 3xTF32 (kept for the measurement: slower than 0 at 8 M atoms)
 *   2  tcgen05.mma 3xTF32, accumulators in tensor memory, block-synchronous (kept for the measurement)
 *   3  tcgen05.mma 3xTF32 -- the default where it applies: k_angular_tc (one thread per atom, <= 56 neurons; software-
 *      pipelined over two 128-atom tiles) or k_angular_split_tc (four lanes per atom, 16-entry slices, <= 104 neurons)
 * (north_star: "tensor cores only for the per-atom descriptor x W0 layer and only if ncu shows it beats CUDA-core
 * FMA": DESIGN.md section 9, profiles/r2_nn_tensor.md).  NEPZBL_NN=ffma|mma|tcsync|tc overrides the default. */
int nep_zbl_network_mode(const nepzbl_handle *h);

/* Counts of the last evaluation / MD step (host outputs, any may be NULL): atoms with a neighbour inside the ZBL
 * range (evaluated by the fp64 pair kernel, Eq. 2-4), and atoms whose angular network inputs |s_nu q_nu| exceeded the
 * fp32 accuracy threshold and were re-evaluated in fp64 (none in a thermal crystal, the
 * disordered core of a cascade; the environment variable NEPZBL_DENSE_THRESHOLD, read at create, overrides the
 * thresholds -- 8 on the 3-body inputs, 3 on the 4-/5-body inputs -- with one number or "t3,t4"; "off" disables
 * the pass). */
int nep_zbl_last_counts(nepzbl_handle *h, int64_t *n_zbl_atoms, int64_t *n_fp64_atoms);

/* Number of kernel launches issued by this handle so far (for bench.py's gpu_launches). */
int64_t nep_zbl_launch_count(const nepzbl_handle *h);

/*
 * Measurement aids (bench.py).  nep_zbl_profile(h, 1) makes every following evaluation / MD step
 * record CUDA events on the launch stream around each kernel group; nep_zbl_profile_read
 * synchronises, sums the elapsed milliseconds and span counts per group into ms[]/counts[]
 * (NEPZBL_PROFILE_SLOTS entries: 0 integrator first half (k_kick_drift incl. the step's book-keeping, and the
 * thermostat's first half-step if set), 1 list rebuild chain, 2 k_radial, 3 the angular kernel (k_angular_tc / k_angular_nn / k_angular_nn_split, see nep_zbl_network_mode), 4 k_force (incl. the
 * second half-kick in its epilogue), 5 k_zbl, 6 the thermostat's second half-step, 7 k_site_fp64) and resets them.
 * nep_zbl_ffma_peak measures the FP32 FMA issue rate of the device (TFLOP/s, 2 flop per FMA) with a
 * register-only microbenchmark, the denominator of the "alu" roofline.
 */
#define NEPZBL_PROFILE_SLOTS 8
int nep_zbl_profile(nepzbl_handle *h, int enable);
int nep_zbl_profile_read(nepzbl_handle *h, double *ms, int64_t *counts);
int nep_zbl_ffma_peak(nepzbl_handle *h, double *tflops);

/*
 * Allocation-free total energies (the reduction of md_energies: E_pot = sum_i U_i, E_kin = sum_i m_i |v_i|^2 / 2 in eV;
 * the NVE / NVT bookkeeping of a cascade run) for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, serving loops, harnesses that forbid it.  The call allocates NOTHING (no cudaMalloc / cudaFree, no
 * allocating library routine, no handle, no workspace): the block partial sums live in a file-scope device array of
 * the library (csrc/no_alloc.cu, 128.25 KiB), which every GPU that loads libnepzbl.so holds until the process exits.
 *   n_atoms     0 .. NEPZBL_STATIC_MAX_ATOMS (the size the array is laid out for); more: NEPZBL_E_UNSUPPORTED.
 *   dev_vel     device, fp64 SoA [3 * n_atoms] (A/fs);  dev_energy  device, fp64 [n_atoms] (eV), e.g. nep_zbl_compute's
 *   dev_types   device, int32 [n_atoms] or NULL (all type 0; required when n_types > 1); values are clamped to the range
 *   host_mass   HOST, n_types doubles (amu), 1 <= n_types <= NEPZBL_STATIC_MAX_TYPES
 *   dev_out     device, 2 doubles: {E_pot, E_kin}, written by the kernel -- valid once the stream reaches that point
 *   stream      cudaStream_t (NULL: the default stream); the call is ASYNCHRONOUS and does not synchronise
 *   host_err    HOST buffer for the error text, or NULL; host_err_len its size
 * All device buffers must belong to the CURRENT device (checked for dev_out: NEPZBL_E_INVALID_ARG otherwise).
 * Fixed-order fp64 sums: repeated calls on the same data give the same bits; against md_energies (another summation
 * tree) the totals agree to rounding (~1e-15 relative).
 * SHARED STATE: every call on a device uses the same array, and the array keeps the last call's contents (the one
 * word that must start at zero is cleared by every call).  Calls issued to ONE stream are safe in any number; two
 * calls that can overlap on the same GPU (different streams, different threads, different processes do NOT share it)
 * RACE on the array and give wrong sums -- order them with an event.
 */
#define NEPZBL_STATIC_MAX_ATOMS 33554432
#define NEPZBL_STATIC_MAX_TYPES 8
int nep_zbl_energy_sums_static(int64_t n_atoms, const double *dev_vel, const double *dev_energy,
                               const int32_t *dev_types, int32_t n_types, const double *host_mass,
                               double *dev_out, void *stream, char *host_err, size_t host_err_len);

#ifdef __cplusplus
}
#endif
#endif /* NEPZBL_H */
