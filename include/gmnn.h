/*
 * gmnn.h -- C ABI of the B200-native GMNN energy-and-force path (arxiv 2505.22168, "apax").
 *
 * One shared library, libgmnn_b200.so (sm_100a only).  Plain pointers and sizes: no torch types,
 * no exceptions across the boundary.  Every pointer is marked HOST or DEVICE.  PyTorch (or any
 * other allocator) owns the caller-facing buffers and the stream; the library owns the model
 * copy, the neighbour list and every workspace inside its two opaque handles.
 *
 * What the path computes (PAPER.md = /root/reference/PAPER.md, the text of the paper):
 *   E(S) = sum_i E_i(G_i)                                              PAPER.md:46  (Eq. 1)
 *   Psi_{i,L,s} = sum_{j != i} R_{Zi,Zj,s}(r_ij) rhat_ij^{(x)L}, L=0..3    PAPER.md:51  (Eq. 2)
 *   G_i = full contractions of the Psi (360 invariants at n_radial=5)  PAPER.md:54-61 (Eq. 3)
 *   E_i = sigma_{Zi} NN(G_i) + mu_{Zi}                                 PAPER.md:63-65 (Eq. 4)
 *   F = -dE/dR (analytic backward, hand-derived)
 *   shallow-ensemble mean / variance over last-layer heads             PAPER.md:75-88 (Eq. 5, 6)
 *   NVE velocity Verlet with a Verlet-skin neighbour list
 * Constants the paper leaves open (Gaussian centres and width, cosine cutoff, swish, block order
 * of the invariants, ...) are the readings R1-R24 of DESIGN.md section 3; each is a field below.
 *
 * Units: Angstrom, eV, fs, amu.  a = F/m * 9.648533212e-3 Ang/fs^2.
 * Cells: cell[9] row-major, rows = lattice vectors a, b, c; any non-singular lattice with a positive diagonal
 * (orthorhombic boxes: off-diagonals 0; sheared / triclinic cells, take the same calls).
 *
 * Return value of every int function: 0 (GMNN_OK) or a negative gmnn_status; the message of the
 * last failure on the calling thread is gmnn_last_error().  Calls are asynchronous on the given
 * stream unless stated otherwise.  There is no CPU fallback: without a CUDA device every compute
 * call returns GMNN_CUDA_ERROR.
 */
#ifndef GMNN_B200_H
#define GMNN_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gmnn_model gmnn_model;   /* hyper-parameters + device copy of the weights        */
typedef struct gmnn_system gmnn_system; /* N atoms, species, neighbour list, all workspaces      */

typedef enum {
    GMNN_OK = 0,
    GMNN_INVALID_ARG = -1,       /* null pointer, N <= 0, r_cut != model's, non-finite input       */
    GMNN_UNSUPPORTED = -2,       /* l_max != 3, triclinic cell, n_radial / n_basis the kernels lack */
    GMNN_NEIGHBOR_OVERFLOW = -3, /* list capacity exceeded where it cannot be regrown (inside MD) */
    GMNN_STALE_NEIGHBORS = -4,   /* an atom moved > skin/2 since the list was built               */
    GMNN_CUDA_ERROR = -5,
    GMNN_OOM = -6,
    GMNN_OUT_OF_BOX = -7         /* a position handed to build_neighbors is outside [0, L)        */
} gmnn_status;

/* How the per-atom MLP (the one dense contraction of the path) is evaluated. */
typedef enum {
    GMNN_MLP_FP32 = 0,   /* fp32 FMA on the SIMT pipes; the fp32-tolerance path                      */
    GMNN_MLP_3XTF32 = 1, /* tcgen05 TF32 tensor cores, 3-term error-compensated split (fp32 tol.)   */
    GMNN_MLP_TF32 = 2,   /* tcgen05 TF32 single pass, operands truncated by the tensor core: measured
                            1e-2 .. 2.5e-2 on the force measure, i.e. NOT within the 2e-3 of a claimed
                            reduced-precision variant; an unclaimed fast mode       */
    GMNN_MLP_3XF16 = 3   /* tcgen05 FP16 tensor cores, the same 3-term split on operands scaled by a
                            power of two from each matrix's absolute maximum (fp32 tol.; twice the
                            MMA rate of 3XTF32)                                                     */
} gmnn_mlp_precision;

/* How F_i = sum_j g_ij - sum_j g_ji is formed.  Both are atomics-free and bit-reproducible. */
typedef enum {
    GMNN_FORCE_GATHER = 0, /* each centre recomputes g_ji from the neighbour's adjoint A_j           */
    GMNN_FORCE_PAIRBUF = 1 /* g_ij evaluated once per directed pair and stored into the neighbour's row
                              through a reverse-pair index that gmnn_build_neighbors (and every
                              in-loop rebuild) builds; rows summed in slot order.  Costs 18 bytes per
                              neighbour slot of device memory, about halves the pair backward          */
} gmnn_force_mode;

typedef struct {
    int32_t n_species;     /* S, 1..8                                                              */
    int32_t n_basis;       /* Gaussians per pair, 1..16 (configs: 7)                               */
    int32_t n_radial;      /* radial channels s (configs: 5; kernels are instantiated for 5)       */
    int32_t l_max;         /* must be 3                                                            */
    float r_cut;           /* Ang                                                                  */
    float r_min;           /* Ang; Gaussian centres r_min + k (r_cut - r_min)/(n_basis - 1)  (R1)  */
    float gauss_gamma;     /* Ang^-2; <= 0 selects 1/(2 Delta^2), Delta = centre spacing     (R2)  */
    int32_t n_hidden;      /* hidden layers, 1..4 (configs: 2)                                     */
    int32_t hidden[4];     /* widths, multiples of 16, <= 1024 (configs: 512, 512)                 */
    int32_t n_heads;       /* 1, or N_ens <= 64 for the shallow ensemble        */
    int32_t n_weight_sets; /* 1 = one NN for all species (Eq. 4); n_species = one NN per
                              species ("the per-species atomic MLP"): atom i uses the (W, b) of set Z_i       */
    int32_t mlp_precision; /* gmnn_mlp_precision                                                   */
    int32_t force_mode;    /* gmnn_force_mode                                                      */
    int32_t radial_basis;  /* 0: equidistant Gaussians; 1: the non-orthogonal Bessel-like functions of Kocer et
                              al. (reading R30; r_min and gauss_gamma are then unused):
                              f_n(r) = (-1)^n sqrt(2) pi / r_cut^1.5 (n+1)(n+2) / sqrt((n+1)^2 + (n+2)^2)
                                       [sinc((n+1) pi r / r_cut) + sinc((n+2) pi r / r_cut)], n = 0 .. n_basis-1 */
    int32_t zbl;           /* 1: add the Ziegler-Littmark-Biersack repulsion (reading R31) per pair,
                              V = zbl_scale k_e Z1 Z2 / r phi(r / a) 1/2 [1 + cos(pi r / zbl_r_max)], r < zbl_r_max */
    float zbl_r_max;       /* Ang, 0 < zbl_r_max <= r_cut                                          */
    float zbl_scale;       /* dimensionless                                                        */
} gmnn_hparams;

typedef struct {            /* HOST pointers, row-major, caller-owned, copied by gmnn_create       */
    const float *beta;      /* [S][S][n_radial][n_basis], centre species first               (R5)  */
    const float *W[5];      /* layer l: [n_weight_sets][fan_in][fan_out], set-major; fan_in(0) = n_features,
                               last fan_out = n_heads                                              */
    const float *b[5];      /* layer l: [n_weight_sets][fan_out]                                   */
    const float *scale;     /* [S] sigma_Z                                                         */
    const float *shift;     /* [S] mu_Z                                                            */
    const float *atomic_numbers; /* [S] nuclear charges for the ZBL term; may be NULL when zbl == 0 */
} gmnn_weights;

/* Number of invariants G_i for n_radial channels (360 at 5), blocks 0-7. */
int32_t gmnn_n_features(int32_t n_radial);

/* Validates the hyper-parameters, copies the weights to the current CUDA device (plus the
 * transposed / split copies the kernels want).  Synchronous.  *out is written only on success. */
int gmnn_create(const gmnn_hparams *hp, const gmnn_weights *w /*HOST*/, gmnn_model **out);
void gmnn_destroy(gmnn_model *m);

/* A system of n_atoms atoms with fixed species (HOST int32 [n_atoms], values 0..S-1).  Allocates
 * the per-atom workspaces; the neighbour list is allocated by the first gmnn_build_neighbors.
 * The model must outlive the system.  Synchronous. */
int gmnn_system_create(const gmnn_model *m, int64_t n_atoms, const int32_t *species /*HOST*/, gmnn_system **out);
void gmnn_system_destroy(gmnn_system *s);

/* Tuning / diagnostics knobs (never needed for correctness):
 *   "lanes_per_atom"  1,2,4,8,16,32: lanes that share one centre atom in the pair kernels (0 = auto)
 *   "ensemble_batch"  0 (default: as many as 4 GB of batch buffers hold) .. 64: heads per batch of the shallow-ensemble
 *                     backward at most (1 = head by head)
 *   "profile"         1: record a CUDA event after every stage of every later energy_forces / md call
 *                     (gmnn_stage_times); setting it (to 0 or 1) discards what was recorded
 *   "md_continue"     1: a gmnn_md_verlet_steps call whose positions and velocities are exactly the
 *                     output of the previous call reuses that call's final forces and energies
 *                     instead of evaluating them again at entry (the caller asserts this)
 *   "md_graph"        1 (default): gmnn_md_verlet_steps captures one step as a CUDA graph after the first
 *                     step and replays it (runs of >= 4 steps, not while "profile" is on); 0: eager loop.
 *                     Results are bit-identical either way
 *   "ef_graph"        1 (default): gmnn_energy_forces (and the _host entry) captures the launches between the gather of the
 *                     caller's positions and the scatter to the caller's outputs as a CUDA graph at the second call of an
 *                     unchanged configuration and replays it afterwards (any gmnn_system_set_int, gmnn_build_neighbors or
 *                     gmnn_system_set_udd_bias call drops it; not while "profile" is on, not for virial calls); 0: eager
 *                     launches.  Results are bit-identical either way
 *   "capacity"        neighbour slots per atom for the next build (0 = estimate from the density)
 *   "mlp_precision", "force_mode": override the model's value for this system; changing force_mode
 *                     invalidates the neighbour list (call gmnn_build_neighbors again)
 *   "tc_pair"         1 (default): 3xTF32 GEMMs on CTA pairs (cta_group::2); 0: single CTAs (3xFP16: always pairs)
 *   "tc_split_bk"     16 | 32 (default): K extent of one pipeline stage of the 3xTF32 GEMM
 *   "tc_flush_k"      multiple of 16 (default 128): K extent after which the FORWARD GEMMs of the 3xTF32 / 3xFP16 modes
 *                     drain the tensor-memory accumulator of the hi.hi products into registers (the tensor core
 *                     accumulates with truncation; the forward GEMMs enter the energies)
 *   "tc_flush_k_bwd"  the same for the BACKWARD GEMMs (default 256; they enter the forces only)
 *   "tc_h_bk"         32 | 64 (default): K extent of one pipeline stage of the 3xFP16 GEMM
 *   "tc_fwd_scheme"   accumulator scheme of the forward 3xFP16 / 3xTF32 GEMMs: 2 (default) = chunks of tc_flush_k alternate between
 *                     two tensor-memory buffers, all cross terms of a chunk issued before its hi.hi terms; 1 = cross terms of the whole
 *                     tile in an accumulator of their own, hi.hi terms drained every tc_flush_k (also taken when a chunk does not
 *                     fit the stage ring)
 *   "tc_tile_order"   0..3: bit 0 forward GEMMs, bit 1 backward GEMMs: 0 (default) = tiles dealt round-robin to the CTA pairs,
 *                     1 = a pair runs the column tiles of one row tile back to back
 *   "tc_dmul_prefetch" -1 (never), 0 (default) .. 64: the backward GEMM prefetches a tile's multiplier block into L2 this many
 *                     pipeline stages before the tile's last
 *   The tc_* knobs are process-wide.  (Builds with -DGMNN_EXPERIMENTS add "tc_debug" and "cb_halves", knock-out
 *   and superseded-variant switches for timing studies; the shipped library rejects them as unknown keys.)
 * Returns GMNN_INVALID_ARG for an unknown key or value. */
int gmnn_system_set_int(gmnn_system *s, const char *key, int64_t value);
int gmnn_system_get_int(const gmnn_system *s, const char *key, int64_t *value /*HOST*/);

/* PAPER.md:169-171, 381 (neighbour list with skin `dr_threshold`, several images in small cells).
 * Builds the full (both directions) Verlet list of all (i, j, n) with |x_j - x_i + n1 a + n2 b + n3 c| < r_cut +
 * skin, n the integer image vector, by a cell list (>= 3 slabs of r_cut + skin between the cell faces of every
 * periodic axis) or an all-pairs image loop (smaller boxes, n_atoms <= 16384).  The membership predicate is
 * evaluated in unfused fp32 exactly as DESIGN.md reading R20 writes it (three-term lattice shift for a general
 * cell), so the set is reproducible bit for bit.  positions: DEVICE float [n_atoms][3], already inside the cell
 * (orthorhombic: [0, L) on every axis, periodic or not; general lattice: fractional coordinates in [0, 1));
 * cell: HOST float[9]; pbc: HOST int32[3]; r_cut must equal the model's.  Synchronises the stream once
 * (capacity check; regrows and retries on overflow). */
int gmnn_build_neighbors(gmnn_system *s, const float *positions /*DEVICE*/, const float cell[9] /*HOST*/,
                         const int32_t pbc[3] /*HOST*/, float r_cut, float skin, void *cuda_stream);

/* Parity hook: the list as (i, j, n) triples in the caller's atom numbering, sorted by
 * (i, j, nx, ny, nz).  Pass i = j = image = NULL to query *n_pairs.  HOST outputs
 * (i, j: int32 [n_pairs]; image: int32 [n_pairs][3]).  Synchronous. */
int gmnn_get_neighbors(gmnn_system *s, int64_t *n_pairs /*HOST*/, int32_t *i, int32_t *j, int32_t *image);

/* The same for the rows of n_sel chosen atoms only (HOST int32 atoms[n_sel], caller numbering): the parity hook
 * for boxes whose whole list is too large to sort on the host.  Synchronous. */
int gmnn_get_neighbor_rows(gmnn_system *s, int64_t n_sel, const int32_t *atoms /*HOST*/, int64_t *n_pairs /*HOST*/,
                           int32_t *i, int32_t *j, int32_t *image);

/* Eq. 1-4 and the analytic forces on the existing list (pairs with r >= r_cut contribute exactly
 * 0).  positions must be a continuous displacement of those the list was built from (atoms are
 * NOT re-wrapped between builds: the list stores image vectors); an atom that moved more than
 * skin/2 raises GMNN_STALE_NEIGHBORS at the next synchronising call (gmnn_check).
 *   positions       DEVICE float [n_atoms][3]
 *   energy          DEVICE double[1]            total E, accumulated in fp64 in a fixed order
 *   energy_per_atom DEVICE float [n_atoms]      nullable
 *   forces          DEVICE float [n_atoms][3]
 * With n_heads > 1 this evaluates the mean energy over the heads and its gradient (PAPER.md:83-86,
 * the cheap force mode of Eq. 6). */
int gmnn_energy_forces(gmnn_system *s, const float *positions, double *energy, float *energy_per_atom,
                       float *forces, void *cuda_stream);

/* The same evaluation plus the virial ("the gradient of the energy with respect to
 * positions and the strain tensor allow the prediction of forces and virials"):
 *   virial  DEVICE double[9], row-major W[a][b] = -sum over directed pairs (i, j, n) of d_a g_b, d = x_j - x_i + n h,
 *           g = dE/dd of the pair, = -dE/d(strain); symmetric up to rounding; stress = -W / V.  Summed from per-atom
 *           terms in fp64 in a fixed order (bit-reproducible).  The first call allocates 36 bytes per atom.
 * With n_heads > 1 it is the virial of the mean energy (and of the UDD-biased energy while a bias is set). */
int gmnn_energy_forces_virial(gmnn_system *s, const float *positions, double *energy, float *energy_per_atom,
                              float *forces, double *virial, void *cuda_stream);

/* The same call with HOST buffers (pinned memory recommended): copies positions in and energy,
 * energy_per_atom (nullable), forces out on the stream, then synchronises it.  This is the
 * end-to-end entry bench.py's `e2e` times. */
int gmnn_energy_forces_host(gmnn_system *s, const float *positions /*HOST*/, double *energy /*HOST*/,
                            float *energy_per_atom /*HOST*/, float *forces /*HOST*/, void *cuda_stream);

/* Eq. 5 (1/N_ens divisor) and Eq. 6, expensive mode: one forward, one backward per head.
 *   e_mean, e_var  DEVICE float [n_atoms]       over the heads' atomic energies
 *   f_mean, f_var  DEVICE float [n_atoms][3]    over the heads' forces, per atom and component
 * Means first, then squared deviations (Welford update in head order), never E[x^2] - E[x]^2. */
int gmnn_ensemble_energy_forces(gmnn_system *s, const float *positions, float *e_mean, float *e_var,
                                float *f_mean, float *f_var, void *cuda_stream);

/* n_steps of velocity Verlet (NVE; NVT while gmnn_system_set_nose_hoover is set) (BASELINE.json configs 2, 5; dt PAPER.md:367), whole loop on the
 * device: kick, drift, skin test, list rebuild when any atom moved > skin/2 since the last build
 * (positions are wrapped into [0, L) at each rebuild, and only then), energy+forces, kick.
 *   positions, velocities  DEVICE float [n_atoms][3], in-out (Ang, Ang/fs)
 *   masses                 DEVICE float [n_atoms] (amu)
 *   epot_series, ekin_series  DEVICE double [n_steps + 1], nullable; index 0 = state at entry
 *   n_rebuilds             HOST int32*, nullable
 * On a model with several heads the energy integrated is their mean (left-hand side of Eq. 6).
 * Needs a list built by gmnn_build_neighbors (its cell, pbc and skin are reused).  Synchronises
 * the stream at the end; returns GMNN_NEIGHBOR_OVERFLOW if an in-loop rebuild ran out of slots
 * (results are then invalid; raise "capacity" and retry). */
int gmnn_md_verlet_steps(gmnn_system *s, float *positions, float *velocities, const float *masses, float dt_fs,
                         int32_t n_steps, double *epot_series, double *ekin_series, int32_t *n_rebuilds,
                         void *cuda_stream);

/* Switching-mode shallow-ensemble MD ("switch between the two modes
 * during a simulation ... the more expensive force uncertainty evaluation is only performed every N
 * steps"; stopping criterion PAPER.md:71; Eq. 5, 6).  Velocity Verlet as gmnn_md_verlet_steps on the
 * MEAN energy of the heads (one backward pass per step).  After steps sampling_rate, 2 sampling_rate, ...
 * the full ensemble pass of gmnn_ensemble_energy_forces runs at the current positions and sample k gets
 *   sigma_e_series[k]     = sqrt(1/M sum_m (E^(m) - mean)^2), E^(m) = sum_i E_i^(m) (fp64 sums, fixed order)
 *   sigma_f_max_series[k] = max_i sqrt(f_var[i][x] + f_var[i][y] + f_var[i][z])
 * The run ends after a sample with sigma_f_max > f_sigma_stop when f_sigma_stop > 0 (<= 0: never stops).
 * The samples do not change the trajectory (bit for bit).
 *   positions, velocities, masses, epot_series, ekin_series   as gmnn_md_verlet_steps (DEVICE); the series
 *                          are valid up to index *n_steps_done
 *   sigma_e_series, sigma_f_max_series   HOST double [n_steps / sampling_rate] (the stream is synchronised
 *                          at every sample to take the stopping decision)
 *   f_var_last             DEVICE float [n_atoms][3], nullable: force variance of the last sample
 *   n_steps_done, n_samples, n_rebuilds   HOST int32*, nullable
 * Works for n_heads = 1 too (all sigma = 0).  Errors as gmnn_md_verlet_steps. */
int gmnn_md_ensemble_steps(gmnn_system *s, float *positions, float *velocities, const float *masses, float dt_fs,
                           int32_t n_steps, int32_t sampling_rate, float f_sigma_stop, double *epot_series,
                           double *ekin_series, double *sigma_e_series, double *sigma_f_max_series, float *f_var_last,
                           int32_t *n_steps_done, int32_t *n_samples, int32_t *n_rebuilds, void *cuda_stream);

/* NVT with a Nose-Hoover chain (PAPER.md:365-375 `thermostat_chain`: chain_length 3,
 * chain_steps 2, sy_steps 3, tau 100 [time steps]).  While set, every step of gmnn_md_verlet_steps and
 * gmnn_md_ensemble_steps applies the Martyna-Tuckerman-Tobias-Klein chain operator for dt/2 before and after the
 * velocity-Verlet step, on the device (the step still replays as a CUDA graph).  Q_0 = 3 N kT tau^2, Q_k = kT tau^2.
 *   temperature_K <= 0 switches the thermostat off (NVE); tau_fs > 0 in fs; 1 <= chain_length <= 8;
 *   1 <= chain_steps <= 16; sy_steps in {1, 3, 5} (Suzuki-Yoshida).  Setting it resets the chain (xi = p_xi = 0). */
int gmnn_system_set_nose_hoover(gmnn_system *s, float temperature_K, float tau_fs, int32_t chain_length,
                                int32_t chain_steps, int32_t sy_steps);
/* Chain state: xi, p_xi HOST double [chain_length] (p_xi in eV fs), and the thermostat's energy
 * sum p_xi^2 / 2Q + 3 N kT xi_0 + kT sum_{k>0} xi_k (eV): epot + ekin + it is conserved.  Synchronises. */
int gmnn_system_get_nose_hoover(gmnn_system *s, double *xi /*HOST*/, double *p_xi /*HOST*/,
                                double *thermostat_energy /*HOST*/, void *cuda_stream);

/* Langevin dynamics for both MD entries, BAOAB splitting: half kick, half
 * drift, v <- c1 v + sqrt(kT (1 - c1^2) / m) xi with c1 = exp(-gamma dt), half drift, forces, half kick.  xi are
 * standard normals from a counter-based generator (splitmix64 outputs (step N + i) 2 + {0, 1} of the stream
 * started at `seed`, Box-Muller in fp64; reading R29), so a trajectory is a function of (seed,
 * first_step) alone and replays as a CUDA graph; `step` counts MD steps from first_step on (device-side).
 *   temperature_K <= 0 switches it off; gamma_per_fs >= 0.  Not together with a Nose-Hoover chain. */
int gmnn_system_set_langevin(gmnn_system *s, float temperature_K, float gamma_per_fs, uint64_t seed, uint64_t first_step);

/* Temperature schedule for whichever thermostat is set ("temperature profiles
 * oscillating between 300 K and 600 K"; reading R32): the target of MD step n (0-based, counted on the device
 * from this call on, over both MD entries) is piecewise linear through the points (steps[k], temperatures_K[k]), constant
 * before the first and after the last.  Both chain half steps of a Nose-Hoover step and the noise of a Langevin step take
 * T(n); the chain masses Q stay those of gmnn_system_set_nose_hoover's temperature.  HOST arrays, 1 <= n_points <= 64,
 * steps strictly ascending from >= 0; n_points = 0 removes the schedule.  The step still replays as a CUDA graph. */
int gmnn_system_set_temperature_schedule(gmnn_system *s, int32_t n_points, const int64_t *steps /*HOST*/,
                                         const float *temperatures_K /*HOST*/);

/* Uncertainty-driven-dynamics bias (Eq. 9) on a model with several
 * heads:  E_b = A [exp(-sigma_E^2 / (N_ens N_atoms B^2)) - 1],  sigma_E^2 = 1/N_ens sum_m (E^(m) - mean)^2 of the
 * heads' TOTAL energies (Eq. 5).  While A != 0, gmnn_energy_forces, gmnn_energy_forces_host, gmnn_md_verlet_steps and
 * gmnn_md_ensemble_steps return the energy mean + E_b and its forces (one backward pass with head weights
 * 1/M + E_b' 2/M (E^(m) - mean)); per-atom energies stay the unbiased mean; gmnn_ensemble_energy_forces and the
 * uncertainty samples are never biased.  A, B in eV; A = 0 switches the bias off (B is then ignored); B > 0.
 * No effect on single-head models (sigma_E = 0). */
int gmnn_system_set_udd_bias(gmnn_system *s, float A, float B);
/* E_b and sigma_E^2 of the latest biased evaluation (zeros if it was not biased); HOST doubles; synchronises. */
int gmnn_system_get_udd_bias(gmnn_system *s, double *e_bias /*HOST*/, double *var_e /*HOST*/, void *cuda_stream);

/* Synchronises the stream and reports a deferred device-side condition (GMNN_STALE_NEIGHBORS,
 * GMNN_NEIGHBOR_OVERFLOW, GMNN_OUT_OF_BOX) or GMNN_OK, clearing it. */
int gmnn_check(gmnn_system *s, void *cuda_stream);

/* Stage timing since "profile" was last set to 1: CUDA events recorded on each call's own stream
 * after every stage (a stage is one kernel, or the few launches named in DESIGN.md section 5).
 * Synchronises on the last event.  Writes, for up to max_stages distinct stage names in order of
 * first appearance, the name, the MEAN duration of one occurrence (ms) and (counts nullable) the
 * number of occurrences; returns the number of names (or a negative status). */
int gmnn_stage_times(gmnn_system *s, int32_t max_stages, const char **names /*HOST*/, float *ms /*HOST*/,
                     int32_t *counts /*HOST*/);

/* Parity hook for the stage tests: copies an internal per-atom array of the last call to HOST,
 * rows in the library's internal (cell-sorted) atom order; "perm" gives internal row -> caller
 * index.  Names: "perm" int32[N]; "psi" float[N][n_radial*20]; "G" float[N][F]; "dG" float[N][F]
 * (without the sigma_Z factor); "A" float[N][n_radial*20]; "count" int32[N].  bytes must match.
 * Synchronous. */
int gmnn_debug_read(gmnn_system *s, const char *name, void *dst /*HOST*/, int64_t bytes);

/* Calibration for bench.py's roofline: the fp32 FMA rate (TFLOP/s, 2 flop per FMA) the current device sustains now, from
 * a register-only kernel of independent FMA chains on every SM (about 10 ms; best of three).  HOST double.  Synchronises. */
int gmnn_measure_fp32_peak(double *tflops /*HOST*/, void *cuda_stream);

/* Total energy without any allocation (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops): *energy = sum_i e_atom[i] in fp64, by the same two fixed-order reduction kernels that produce the total
 * energy of gmnn_energy_forces (Eq. 4: E = sum_i E_i), so the result depends on
 * n_atoms only, never on scheduling.  e_atom: DEVICE float[n_atoms] (e.g. the e_atom output of gmnn_energy_forces);
 * energy: DEVICE double[1]; both owned by the caller, on the current device; asynchronous on `cuda_stream`.
 * The block partials live in a file-scope device array of the library (8 KB, held by every GPU that loads the library
 * until exit), which sets the limit n_atoms <= GMNN_STATIC_SUM_MAX_ATOMS: more returns GMNN_INVALID_ARG with a message
 * and launches nothing.  The call makes no cudaMalloc / cudaFree and no allocating library call.  All calls share that
 * array: calls that overlap on the GPU (different streams or host threads) race; calls in stream order do not, and no
 * call reads what an earlier one left (every slot read is written first by the same call). */
#define GMNN_STATIC_SUM_MAX_ATOMS 16777216
int gmnn_sum_energies_static(const float *e_atom /*DEVICE*/, int64_t n_atoms, double *energy /*DEVICE*/, void *cuda_stream);

/* Number of kernel launches issued by this library since it was loaded (bench.py's gpu_launches). */
int64_t gmnn_launch_count(void);

/* Thread-local message for the last non-zero return. */
const char *gmnn_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GMNN_B200_H */
