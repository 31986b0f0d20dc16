// gmnn_internal.h -- handles, device buffers and kernel launchers shared by the .cu files of
// libgmnn_b200.so.  Nothing here is visible through the C ABI (include/gmnn.h).
#pragma once

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/gmnn.h"

namespace gmnn {

constexpr int MAX_SPECIES = 8;
constexpr int MAX_BASIS = 16;
constexpr int MAX_LAYERS = 5;
constexpr int NBR_J_BITS = 22;  // neighbour entry: j in the low 22 bits, image code above
constexpr uint32_t NBR_J_MASK = (1u << NBR_J_BITS) - 1u;
constexpr int64_t MAX_ATOMS = (int64_t)1 << NBR_J_BITS;
constexpr int SMALL_BOX_MAX_ATOMS = 16384;
constexpr int MAX_STAGE_EVENTS = 1 << 16;
// device scalars of gmnn_system::amax: absolute maxima (fp32 bit patterns) of the 3xFP16 GEMM operands
enum AmaxSlot { AMAX_G = 0, AMAX_H = 1, AMAX_DZ = AMAX_H + MAX_LAYERS, AMAX_BVT = AMAX_DZ + 2, AMAX_D, AMAX_SLOTS };
constexpr int MAX_HEAD_SLOTS = 16;  // partial sums per atom of the head fused into the last GEMM epilogue
constexpr int PSI = 20;  // unique monomials per channel (contraction.cuh NM)

// device-side flag words (int32) in System::flags
enum Flag { FLAG_MAXCOUNT = 0, FLAG_STALE = 1, FLAG_OUT_OF_BOX = 2, FLAG_REBUILDS = 3, FLAG_DISP2 = 4, FLAG_REV_MISSING = 5, FLAG_MD_STEP = 6, FLAG_WORDS = 8 };

void set_error(const char *fmt, ...);
extern long long g_launch_count;
// One-time set-up (function attributes, __constant__ tables) is per DEVICE: the guards are arrays
// indexed by the current device, never process-wide flags (a handle is bound to the device that was
// current at gmnn_create and every call checks it).
constexpr int MAX_DEVICES = 64;
inline int current_device() {
    int d = 0;
    cudaGetDevice(&d);
    return (d >= 0 && d < MAX_DEVICES) ? d : 0;
}
#define GMNN_LAUNCHED() (++::gmnn::g_launch_count)

#define GMNN_CUDA(expr)                                                                          \
    do {                                                                                         \
        cudaError_t err__ = (expr);                                                              \
        if (err__ != cudaSuccess) {                                                              \
            ::gmnn::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(err__), __FILE__, __LINE__); \
            return err__ == cudaErrorMemoryAllocation ? GMNN_OOM : GMNN_CUDA_ERROR;              \
        }                                                                                        \
    } while (0)

struct Geometry {  // passed by value to kernels
    float L[3];        // orthorhombic edge lengths = the diagonal of h
    float invL[3];
    int pbc[3];
    int ncell[3];
    float inv_edge[3];  // orthorhombic: cells per Angstrom (ncell / L)
    int kimg[3];  // image range of the small-box path
    float r_list2;
    float r_cut2;  // rows are built inside-r_cut first, skin shell last (neighbor.cu)
    // general lattice: h rows = lattice vectors a, b, c; fractional s = x . hinv.  triclinic = 0
    // when every off-diagonal element is zero: the kernels then take the orthorhombic expressions, whose results
    // the general ones reproduce bit for bit (adding an exact zero), so one list format serves both.
    int triclinic;
    float h[9];
    float hinv[9];
};

// lattice shift of image (n1, n2, n3), component x: the diagonal term first, so that with zero off-diagonals the
// value is exactly n_x L_x
__device__ __forceinline__ float lattice_shift(const Geometry &g, int x, float n1, float n2, float n3) {
    if (!g.triclinic) return (x == 0 ? n1 : x == 1 ? n2 : n3) * g.L[x];
    return n1 * g.h[x] + n2 * g.h[3 + x] + n3 * g.h[6 + x];
}

struct RadialParams {  // passed by value to the pair kernels
    int n_species, n_basis, kb;  // kb = n_basis rounded up to 4 (row pitch of the beta table)
    float r_cut, r_cut2, inv_rc, r_min, delta, gamma;
    int basis_kind;              // 0 Gaussians, 1 Bessel-like (hparams.radial_basis)
    float bessel_c[MAX_BASIS];   // (-1)^n sqrt(2) pi / r_cut^1.5 (n+1)(n+2) / sqrt((n+1)^2 + (n+2)^2)
    int zbl_on;                  // ZBL repulsion (hparams.zbl)
    float zbl_r_max2, zbl_inv_rmax, zbl_pref;  // r_max^2, 1 / r_max, 1/2 zbl_scale k_e
    float zbl_z[MAX_SPECIES], zbl_zpow[MAX_SPECIES];  // Z and Z^0.23 per species
};

}  // namespace gmnn

struct gmnn_model {
    gmnn_hparams hp;
    int device = 0;            // CUDA device the weights live on (current at gmnn_create)
    int n_features;
    int n_layers;              // n_hidden + 1
    int dims[gmnn::MAX_LAYERS + 1];  // dims[0] = F, hidden..., n_heads
    gmnn::RadialParams rp;
    float *beta = nullptr;     // [S*S][n_radial][kb] zero padded
    // Weight sets (hp.n_weight_sets: 1 = one NN for all species, Eq. 4; n_species = one NN per species): every
    // per-layer array below holds the sets back to back (set-major), set t of layer l at offset t * wsize(l)
    // (bias: t * dims[l + 1]; stacked hi / lo copies: t * 2 * wsize(l)).
    int n_sets = 1;
    size_t wsize(int l) const { return (size_t)dims[l] * dims[l + 1]; }
    float *W[gmnn::MAX_LAYERS] = {};   // [fan_in][fan_out]
    float *WT[gmnn::MAX_LAYERS] = {};  // [fan_out][fan_in]
    // tf32 hi / lo split of the two, stacked: rows [0, R) hold hi = tf32(w), rows [R, 2R) lo = w - hi
    // (the B operands of the 3xTF32 GEMMs of mlp_tc.cu; split once here instead of per tile on chip)
    float *Ws[gmnn::MAX_LAYERS] = {};   // [2 * fan_in][fan_out]
    float *WTs[gmnn::MAX_LAYERS] = {};  // [2 * fan_out][fan_in]
    // fp16 hi / lo split of the two scaled by a power of two (3xFP16, mlp_tc.cu), stacked the same way, and
    // the absolute maximum of each layer's weights (fp32 bit pattern) that fixes the scale
    uint16_t *Wh[gmnn::MAX_LAYERS] = {}, *WTh[gmnn::MAX_LAYERS] = {};
    uint32_t *wmax = nullptr;           // [MAX_LAYERS] device
    float *b[gmnn::MAX_LAYERS] = {};
    float *scale = nullptr, *shift = nullptr;  // [S]
    float *head_mean_w = nullptr;  // [n_heads] = 1/M (device)
    float *w_mean = nullptr;       // per set [H_last + 1]: W_last 1/M and, last, mean(b_last): the mean of the heads as one head
};

struct gmnn_system {
    const gmnn_model *model = nullptr;
    int device = 0;              // = model->device; calls from another current device are rejected
    int64_t N = 0;
    int32_t *species = nullptr;  // caller order (device)
    // geometry of the last build
    bool have_list = false, small_box = false;
    gmnn::Geometry geo{};
    float r_cut = 0.f, skin = 0.f;
    int64_t ncells = 0, ncells_alloc = 0;
    // cell sort
    int32_t *cell_of = nullptr;      // [N] caller order
    int32_t *cell_count = nullptr;   // [ncells + 1]
    int32_t *cell_start = nullptr;   // [ncells + 1]
    int32_t *cell_fill = nullptr;    // [ncells]
    int32_t *slot_tmp = nullptr;     // [N]
    int32_t *perm = nullptr;         // [N] internal -> caller
    float4 *pos4 = nullptr;          // [N] internal order: x y z species(bits)
    float *xref = nullptr;           // [N][3] caller order, positions at build
    // neighbour list
    uint32_t *nbr = nullptr;         // [N][cap]
    int32_t *count = nullptr;        // [N]
    uint16_t *rev = nullptr;         // [N][cap] slot of the reverse pair (GMNN_FORCE_PAIRBUF)
    uint16_t *runs = nullptr;        // [N][56] first slot of each of the 2 x 27 cell runs of a row, and its length
    float4 *gbuf = nullptr;          // [N][cap] g_ij, stored in the row of j at the reverse slot
    bool list_has_rev = false;
    int cap = 0;
    int cap_request = 0;
    // MLP rows.  With one weight set the per-atom matrices of the MLP stage (psi, G, H, D, dZ, dG, A) are in
    // internal atom order: row = atom, n_rows = N, mrow = row_atom = nullptr.  With per-species sets the rows
    // are grouped by species so that every 256-row tile pair of the GEMMs uses ONE weight set: species z owns
    // rows [seg_row0[z], seg_row0[z] + seg_rows[z]) of a segment padded to a multiple of 256 (padding rows keep
    // psi = 0 and are never read back); inside a segment atoms keep their internal (cell) order.  mrow[k] = row
    // of internal atom k, row_atom[r] = internal atom of row r or -1; both are rebuilt with the list.
    int64_t n_rows = 0;
    int64_t seg_row0[gmnn::MAX_SPECIES] = {}, seg_rows[gmnn::MAX_SPECIES] = {};
    int32_t *mrow = nullptr, *row_atom = nullptr;
    int32_t *sp_count = nullptr;     // [blocks of 256 atoms][MAX_SPECIES] scratch of the row assignment
    // workspaces (row order)
    float *psi = nullptr, *G = nullptr, *dG = nullptr, *A = nullptr;
    float *H[gmnn::MAX_LAYERS] = {}, *D[gmnn::MAX_LAYERS] = {};
    float *dZ[2] = {};
    float *Bv = nullptr;             // diag(v) W^T of the last hidden layer
    float *BvT = nullptr;            // its transpose: W diag(v), [fan_in][fan_out] (B operand of mlp_tc.cu)
    float *BvTs = nullptr;           // stacked hi / lo split of BvT
    uint16_t *BvTh = nullptr;        // ... in fp16 (3xFP16)
    uint32_t *amax = nullptr;        // [AMAX_SLOTS] absolute maxima of the 3xFP16 GEMM operands (see gmnn::AmaxSlot)
    float *vhead = nullptr;          // [H_last]
    float *head_w = nullptr;         // [n_heads] weights of the differentiated energy
    float *ypart = nullptr;          // [MAX_HEAD_SLOTS][N padded to 128]: partial head sums (mlp_tc.cu EPI_HIDDEN_HEAD)
    double *nhc = nullptr;           // [26] Nose-Hoover chain: xi[8], p_xi[8], Q[8], scale, thermostat energy (lazy)
    int nhc_len = 0, nhc_chain_steps = 2, nhc_sy_steps = 3;  // nhc_len == 0: NVE
    double nhc_kT = 0.0;
    // thermostat target: both thermostats read k_B T (eV) from the device scalar kT_now; a temperature schedule
    // (piecewise linear in the MD step, gmnn_system_set_temperature_schedule) rewrites it at the start of every step
    double *kT_now = nullptr;        // device [1] (lazy)
    int sched_n = 0;                 // points of the schedule (0: constant target)
    int64_t *sched_steps = nullptr;  // device [sched_n]
    float *sched_temps = nullptr;    // device [sched_n] (K)
    uint64_t *sched_step = nullptr;  // device: MD steps since the schedule was set
    bool lang_on = false;            // Langevin (BAOAB) instead of the plain kick + drift
    double lang_gamma = 0.0, lang_kT = 0.0;  // 1/fs, eV
    uint64_t lang_seed = 0;
    uint64_t *lang_step = nullptr;   // device: MD steps since the thermostat was set (counter of the generator)
    float udd_A = 0.f, udd_B = 1.f;  // UDD bias parameters (Eq. 9); active when udd_A != 0 and n_heads > 1
    bool udd_active = false;         // this evaluation adds the bias: e_total[4] = E_b, e_total[5] = sigma_E^2
    bool use_mean_head = false;      // MD on a multi-head model: forward with model->w_mean as the only head
    bool heads_fused = false;        // the last mlp_forward left ypart instead of H[L-1]
    int head_slots = 0;
    float *e_heads = nullptr;        // [N][n_heads]
    float *vir_atom = nullptr;       // [9][N] per-atom virial terms -sum_j d_a g_b (lazy; gmnn_energy_forces_virial)
    bool want_virial = false;        // this evaluation's pair backward also leaves vir_atom
    float *e_zbl = nullptr;          // [N] internal order: sum over the centre's pairs of V_ZBL / 2 (models with zbl)
    float *e_atom = nullptr;         // [N]
    float *f_int = nullptr;          // [N][3]
    float *f_tmp = nullptr;          // [N][3] caller order (ensemble, MD)
    double *partial = nullptr;       // reduction scratch
    double *e_total = nullptr;       // [6] device scalars (epot, ekin, sigma_E, bits of sigma_F,max, E_b, sigma_E^2 of the bias)
    // batched shallow-ensemble backward (gmnn_api.cu ensemble_pass): ens_batch heads per pass in buffers whose row tiles
    // are ordered [atom tile][head]; 0 / 1 outside such a pass.  ens_head: the head the pair backward reads.
    int ens_batch = 0, ens_head = 0, ens_cap = 0;  // ens_cap: heads the buffers below hold
    const float *seed_w = nullptr;  // head weights the kept backward seed (vhead, Bv / BvT, its split and maximum) was prepared for
    int seed_prec = -1;             // ... and the MLP mode
    int ens_batch_max = 0;                          // knob "ensemble_batch": heads per batch at most (0: as many as fit)
    float *ens_dZ[2] = {}, *ens_dG = nullptr, *ens_A = nullptr;
    // pair-buffer force mode: per-head own-direction force sums [heads][3 N] and pair buffers [heads][N cap] of the batch
    // (k_pair_backward_heads); ens_gcap = the list capacity they were sized for
    float *ens_f = nullptr;
    float4 *ens_gbuf = nullptr;
    int ens_gcap = 0, ens_gheads = 0;
    float *ens_BvT = nullptr, *ens_BvTs = nullptr;
    uint16_t *ens_BvTh = nullptr;
    float *ens_scratch = nullptr;    // [11 N] switching-mode samples: kept forces, e_mean, e_var, f_mean, f_var (lazy)
    int32_t *flags = nullptr;        // FLAG_WORDS
    int32_t *flags_host = nullptr;   // pinned
    // knobs
    int lanes_per_atom = 0;
    int profile = 0;
    int md_graph = 1;                // knob: replay the MD step as a CUDA graph (not while profiling stages)
    cudaStream_t graph_stream = nullptr;  // capture / replay stream (the caller's may be the legacy stream)
    // gmnn_energy_forces: the launches between the gather and the output scatter, captured at the second call of an unchanged
    // configuration (gmnn_api.cu forward_backward); knob "ef_graph"
    int ef_graph = 1;
    cudaGraphExec_t ef_exec = nullptr;
    long long ef_gen = 0, ef_seen_gen = 0, ef_launches = 0;
    const float *ef_seed_w = nullptr;  // seed_w (below) at the capture: the graph is valid while the kept seed is the same
    cudaEvent_t graph_ev[2] = {};
    int md_continue = 0;             // knob: the next md call continues the previous one
    bool md_state_valid = false;     // f_tmp / e_total hold the forces and energies of the last md step
    int mlp_precision = 0, force_mode = 0;
    // stage timing
    std::vector<cudaEvent_t> events;
    std::vector<const char *> stage_names;
    int n_stage_events = 0;
    // host staging for the _host entry
    float *stage_pos = nullptr, *stage_f = nullptr, *stage_e = nullptr;
};

namespace gmnn {

// One launch unit of the MLP stage: a run of rows that uses one weight set.  One segment (all rows, set 0)
// with a shared NN; one per non-empty species with per-species sets (rows padded to a multiple of 256).
struct MlpSeg {
    int64_t row0;  // first row (a multiple of 128: a tile boundary of the tile-transposed matrices)
    int64_t rows;  // rows handed to the GEMMs (real rows, or the padded segment)
    int64_t real;  // rows that carry an atom
    int set;
};
inline int mlp_segments(const gmnn_system *s, MlpSeg *seg) {
    if (s->model->n_sets == 1) {
        seg[0] = MlpSeg{0, s->N, s->N, 0};
        return 1;
    }
    int n = 0;
    for (int z = 0; z < s->model->hp.n_species; ++z)
        if (s->seg_rows[z] > 0) seg[n++] = MlpSeg{s->seg_row0[z], (s->seg_rows[z] + 255) / 256 * 256, s->seg_rows[z], z};
    return n;
}
// first element of row block `row0` of a tile-transposed [rows/128][width][128] matrix
template <class T>
inline T *tile_rows(T *base, int64_t row0, int width) {
    return base + (row0 / 128) * (int64_t)width * 128;
}

// neighbor.cu
int launch_build(gmnn_system *s, const float *positions, cudaStream_t st, const int32_t *cond, float thr2,
                 bool wrap_first, float *positions_mut);
int launch_gather_positions(gmnn_system *s, const float *positions, cudaStream_t st, bool check_stale);

// descriptor.cu
int launch_pair_forward(gmnn_system *s, cudaStream_t st);
int launch_contract_forward(gmnn_system *s, cudaStream_t st);
int launch_contract_backward(gmnn_system *s, cudaStream_t st);
int launch_pair_backward(gmnn_system *s, cudaStream_t st);  // dispatches on force_mode
int launch_pair_backward_welford(gmnn_system *s, int head, float *f_mean, float *f_m2, cudaStream_t st);  // a12, one head
int launch_pair_backward_heads_welford(gmnn_system *s, int head_first, int n_heads, float *f_mean, float *f_m2, cudaStream_t st);  // a12, a batch of heads

// mlp_tc.cu
int launch_split_stack(const float *src, float *dst, int64_t n, cudaStream_t st);  // dst[0..n) hi, dst[n..2n) lo
int launch_absmax(const float *src, int64_t n, uint32_t *amax, cudaStream_t st);  // *amax = max |src| (reset first)
int launch_split_stack_h(const float *src, uint16_t *dst, int64_t n, const uint32_t *amax, cudaStream_t st);  // fp16, scaled by *amax

// mlp_simt.cu
int launch_mlp_forward_simt(gmnn_system *s, cudaStream_t st);
int launch_mlp_heads(gmnn_system *s, const float *head_w_dev, cudaStream_t st);
int launch_mlp_seed(gmnn_system *s, const float *head_w_dev, cudaStream_t st);
int launch_mlp_backward_simt(gmnn_system *s, const float *head_w_dev, cudaStream_t st);
int launch_mlp_backward_tc_heads(gmnn_system *s, int head0, int n_heads, cudaStream_t st);  // mlp_tc.cu: heads batched

// md.cu / reductions
int launch_scatter_outputs(gmnn_system *s, float *e_atom_out, float *forces_out, cudaStream_t st);
int launch_energy_sum(gmnn_system *s, double *energy_out, cudaStream_t st, double *energy_out2 = nullptr);
int launch_virial_sum(gmnn_system *s, double *virial_out, cudaStream_t st);  // [9] fixed-order fp64 sums of vir_atom
int launch_kick_drift(gmnn_system *s, float *x, float *v, const float *f, const float *m, float dt, cudaStream_t st);
int launch_kick_ke(gmnn_system *s, float *v, const float *f, const float *m, float dt, double *ekin_out,
                   cudaStream_t st, double *ekin_out2 = nullptr);
int launch_ke(gmnn_system *s, const float *v, const float *m, double *ekin_out, cudaStream_t st,
              double *ekin_out2 = nullptr);
int launch_series_append(gmnn_system *s, double *epot_series, double *ekin_series, cudaStream_t st);
int launch_series_reset(gmnn_system *s, int32_t next_index, cudaStream_t st);
int launch_ensemble_energy_stats(gmnn_system *s, float *e_mean, float *e_var, cudaStream_t st);
int launch_finish_var(int64_t n, float *m2, int n_heads, cudaStream_t st);
int launch_baoab(gmnn_system *s, float *x, float *v, const float *f, const float *m, float dt, cudaStream_t st);
int launch_nhc_half(gmnn_system *s, float *v, double *ek, float dt, cudaStream_t st);
int launch_schedule_eval(gmnn_system *s, cudaStream_t st);
int launch_fma_peak(int blocks, int iters, float *scratch, cudaStream_t st);  // blocks x 256 threads x iters x 128 FMA  // kT_now <- k_B T(step), step += 1
int launch_udd_weights(gmnn_system *s, float *head_w_out, double *scal, cudaStream_t st);
int launch_uncertainty_scalars(gmnn_system *s, const float *f_var, double *out_d, int32_t *out_bits, cudaStream_t st);

}  // namespace gmnn
