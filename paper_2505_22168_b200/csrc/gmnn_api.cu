// gmnn_api.cu -- the C ABI of include/gmnn.h: handles, validation, buffer ownership and the
// order in which the kernels of neighbor.cu / descriptor.cu / mlp_*.cu / md.cu run.
// Every step of the path runs in those kernels; this file only allocates, launches and reports.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <numeric>

#include "contraction.cuh"
#include "gmnn_internal.h"

namespace gmnn {

static thread_local char g_error[512] = "";
long long g_launch_count = 0;

void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
}

int launch_mlp_forward_tc(gmnn_system *s, cudaStream_t st);
extern int g_tc_split_bk, g_tc_flush_k, g_tc_flush_k_bwd, g_tc_pair, g_tc_h_bk, g_tc_tile_order, g_tc_dmul_prefetch, g_tc_fwd_scheme;
#ifdef GMNN_EXPERIMENTS
extern int g_tc_debug, g_cb_halves;
#endif
int launch_mlp_backward_tc(gmnn_system *s, const float *head_w_dev, cudaStream_t st);

// A handle is bound to the device that was current at gmnn_create: per-device state (the weights, the
// kernels' one-time attributes, __constant__ tables) would be silently wrong from another device.
static int check_device(int device, const char *who) {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != device) {
        set_error("%s: the handle belongs to CUDA device %d, the current device is %d", who, device, cur);
        return GMNN_INVALID_ARG;
    }
    return GMNN_OK;
}

template <class T>
static int dev_alloc(T **p, size_t n) {
    *p = nullptr;
    GMNN_CUDA(cudaMalloc((void **)p, sizeof(T) * (n > 0 ? n : 1)));
    return GMNN_OK;
}
template <class T>
static void dev_free(T *&p) {
    if (p) cudaFree((void *)p);
    p = nullptr;
}
template <class T>
static int upload(T **p, const T *host, size_t n) {
    int rc = dev_alloc(p, n);
    if (rc) return rc;
    GMNN_CUDA(cudaMemcpy(*p, host, sizeof(T) * n, cudaMemcpyHostToDevice));
    return GMNN_OK;
}

__global__ void k_set_onehot(int M, int m, float *w) {
    const int t = threadIdx.x;
    if (t < M) w[t] = (t == m) ? 1.f : 0.f;
}

// Stage timing ("profile" = 1): one CUDA event after every stage of every call, on the call's own
// stream, kept until "profile" is set again; gmnn_stage_times averages them per stage name.
struct StageTimer {
    gmnn_system *s;
    cudaStream_t st;
    StageTimer(gmnn_system *s_, cudaStream_t st_) : s(s_), st(st_) {}
    void begin() { mark(nullptr); }
    void mark(const char *name) {
        if (!s->profile || s->n_stage_events >= MAX_STAGE_EVENTS) return;
        if ((int)s->events.size() <= s->n_stage_events) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            s->events.push_back(e);
            s->stage_names.push_back(nullptr);
        }
        s->stage_names[s->n_stage_events] = name;
        cudaEventRecord(s->events[s->n_stage_events++], st);
    }
};

static int mlp_forward(gmnn_system *s, cudaStream_t st) {
    if (s->mlp_precision == GMNN_MLP_FP32) return launch_mlp_forward_simt(s, st);
    return launch_mlp_forward_tc(s, st);
}
static int mlp_backward(gmnn_system *s, const float *head_w, cudaStream_t st) {
    if (s->mlp_precision == GMNN_MLP_FP32) return launch_mlp_backward_simt(s, head_w, st);
    return launch_mlp_backward_tc(s, head_w, st);
}

// Bumped by every call that can change what an evaluation launches (knobs, including the process-wide tc_* ones, a list
// build, the UDD bias): a captured evaluation (below) is replayed only while the value it was captured at stands.
static long long g_config_gen = 1;

// positions -> E_i, F (internal order), for the energy whose head weights are head_w (device).
// allow_graph (gmnn_energy_forces only): everything between the gather of the caller's positions and the scatter to the
// caller's outputs touches library buffers only, so its launches (about 20; what bounds the call below some 10^4 atoms)
// are captured once as a CUDA graph -- at the second call of an unchanged configuration, the first having done the
// one-time set-up eagerly -- and replayed by later calls.  Not while stage events are recorded or a virial is asked for.
static int forward_backward(gmnn_system *s, const float *positions, const float *head_w, bool check_stale,
                            cudaStream_t st, StageTimer &T, bool allow_graph = false) {
    int rc;
    s->udd_active = s->udd_A != 0.f && s->model->hp.n_heads > 1 && head_w == s->model->head_mean_w;
    if (s->udd_active) s->use_mean_head = false;  // the bias needs every head's energy
    if ((rc = launch_gather_positions(s, positions, st, check_stale))) return rc;
    T.mark("gather");
    auto core = [&](cudaStream_t q, StageTimer &TT) -> int {
        int r;
        const float *hw = head_w;
        if (s->mlp_precision == GMNN_MLP_3XF16)  // maxima of G, H, dZ: rebuilt by this evaluation's kernels
            GMNN_CUDA(cudaMemsetAsync(s->amax, 0, sizeof(uint32_t) * AMAX_BVT, q));
        if ((r = launch_pair_forward(s, q))) return r;
        TT.mark("pair_forward");
        if ((r = launch_contract_forward(s, q))) return r;
        TT.mark("contract_forward");
        if ((r = mlp_forward(s, q))) return r;
        TT.mark("mlp_forward");
        if ((r = launch_mlp_heads(s, hw, q))) return r;
        if (s->udd_active) {  // UDD bias: the head weights of the backward come from this forward's head totals
            if ((r = launch_udd_weights(s, s->head_w, s->e_total + 4, q))) return r;
            hw = s->head_w;
        }
        TT.mark("mlp_heads");
        if ((r = mlp_backward(s, hw, q))) return r;
        TT.mark("mlp_backward");
        if ((r = launch_contract_backward(s, q))) return r;
        TT.mark("contract_backward");
        if ((r = launch_pair_backward(s, q))) return r;
        TT.mark("pair_backward");
        return GMNN_OK;
    };
    if (!(allow_graph && s->ef_graph && !s->profile && !s->want_virial)) return core(st, T);
    // (the captured launches rely on the backward seed kept in the system's buffers, mlp_tc.cu launch_mlp_backward_tc: an
    // ensemble pass or a biased evaluation in between overwrites those buffers and clears seed_w)
    if (s->ef_exec && s->ef_gen == g_config_gen && s->seed_w != s->ef_seed_w) {
        cudaGraphExecDestroy(s->ef_exec);
        s->ef_exec = nullptr;
        return core(st, T);  // prepares the seed again; the next call captures
    }
    if (s->ef_exec && s->ef_gen == g_config_gen) {  // replay
        GMNN_CUDA(cudaGraphLaunch(s->ef_exec, st));
        g_launch_count += s->ef_launches;
        return GMNN_OK;
    }
    if (s->ef_exec) {
        cudaGraphExecDestroy(s->ef_exec);
        s->ef_exec = nullptr;
    }
    if (s->ef_seen_gen != g_config_gen) {  // first call of this configuration: eagerly
        s->ef_seen_gen = g_config_gen;
        return core(st, T);
    }
    // second call: capture on the library's own stream (the caller's may be the legacy stream), then launch
    if (!s->graph_stream) {
        GMNN_CUDA(cudaStreamCreateWithFlags(&s->graph_stream, cudaStreamNonBlocking));
        GMNN_CUDA(cudaEventCreateWithFlags(&s->graph_ev[0], cudaEventDisableTiming));
        GMNN_CUDA(cudaEventCreateWithFlags(&s->graph_ev[1], cudaEventDisableTiming));
    }
    const long long launches_before = g_launch_count;
    cudaGraph_t graph = nullptr;
    GMNN_CUDA(cudaStreamBeginCapture(s->graph_stream, cudaStreamCaptureModeThreadLocal));
    rc = core(s->graph_stream, T);
    const cudaError_t cap = cudaStreamEndCapture(s->graph_stream, &graph);
    s->ef_launches = g_launch_count - launches_before;
    g_launch_count = launches_before;
    if (rc || cap != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        if (!rc) {
            set_error("CUDA graph capture of the energy-and-force evaluation failed: %s", cudaGetErrorString(cap));
            rc = GMNN_CUDA_ERROR;
        }
        return rc;
    }
    const cudaError_t ge = cudaGraphInstantiate(&s->ef_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ge != cudaSuccess) {
        s->ef_exec = nullptr;
        set_error("CUDA graph instantiation of the energy-and-force evaluation failed: %s", cudaGetErrorString(ge));
        return GMNN_CUDA_ERROR;
    }
    s->ef_gen = g_config_gen;
    s->ef_seed_w = s->seed_w;
    GMNN_CUDA(cudaGraphLaunch(s->ef_exec, st));
    g_launch_count += s->ef_launches;
    return GMNN_OK;
}

// a12: one forward, then one backward per head with a one-hot head weight; Welford over the heads.
// Uses f_tmp as the per-head force buffer.
static int ensemble_pass(gmnn_system *s, const float *positions, float *e_mean, float *e_var, float *f_mean,
                         float *f_var, cudaStream_t st) {
    const int M = s->model->hp.n_heads;
    int rc;
    struct ProfileOff {  // stage events are not recorded inside the pass; restored on every return path
        gmnn_system *s;
        int keep;
        explicit ProfileOff(gmnn_system *s_) : s(s_), keep(s_->profile) { s->profile = 0; }
        ~ProfileOff() { s->profile = keep; }
    } profile_off(s);
    if ((rc = launch_gather_positions(s, positions, st, true))) return rc;
    if (s->mlp_precision == GMNN_MLP_3XF16)  // operand maxima of this evaluation (as forward_backward does)
        GMNN_CUDA(cudaMemsetAsync(s->amax, 0, sizeof(uint32_t) * AMAX_BVT, st));
    if ((rc = launch_pair_forward(s, st))) return rc;
    if ((rc = launch_contract_forward(s, st))) return rc;
    if ((rc = mlp_forward(s, st))) return rc;
    if ((rc = launch_mlp_heads(s, s->model->head_mean_w, st))) return rc;
    if ((rc = launch_ensemble_energy_stats(s, e_mean, e_var, st))) return rc;
    // Heads batched through the backward GEMMs and the contraction backward (mlp_tc.cu launch_mlp_backward_tc_heads): as many
    // heads per pass as 4 GB of batch buffers hold (at least one); tensor-core split modes with one weight set.  Else head by head.
    const gmnn_model *mdl = s->model;
    const int L = mdl->hp.n_hidden;
    int HB = 1;
    if (M > 1 && mdl->n_sets == 1 && (s->mlp_precision == GMNN_MLP_3XF16 || s->mlp_precision == GMNN_MLP_3XTF32)) {
        int maxw = 0;
        for (int l = 1; l <= L; ++l) maxw = std::max(maxw, mdl->dims[l]);
        const size_t NP = (size_t)((s->N + 127) / 128 * 128);
        const bool pairbuf = s->force_mode == GMNN_FORCE_PAIRBUF && s->list_has_rev;
        const double per_head = (double)NP * (2.0 * maxw + mdl->n_features + mdl->hp.n_radial * PSI) * 4.0 +
                                (pairbuf ? (double)s->N * (16.0 * s->cap + 12.0) : 0.0);
        HB = (int)std::max(1.0, std::min<double>((double)M, std::floor(4.0e9 / per_head)));
        if (s->ens_batch_max > 0 && HB > s->ens_batch_max) HB = s->ens_batch_max;  // knob "ensemble_batch"
        if (HB >= 2 && s->ens_cap < HB) {
            dev_free(s->ens_dZ[0]); dev_free(s->ens_dZ[1]); dev_free(s->ens_dG); dev_free(s->ens_A);
            dev_free(s->ens_BvT); dev_free(s->ens_BvTs); dev_free(s->ens_BvTh);
            s->ens_cap = 0;
            const size_t bv = (size_t)mdl->dims[L] * mdl->dims[L - 1] * HB;
            if ((rc = dev_alloc(&s->ens_dZ[0], NP * HB * maxw)) || (rc = dev_alloc(&s->ens_dZ[1], NP * HB * maxw)) ||
                (rc = dev_alloc(&s->ens_dG, NP * HB * mdl->n_features)) ||
                (rc = dev_alloc(&s->ens_A, NP * HB * mdl->hp.n_radial * PSI)) || (rc = dev_alloc(&s->ens_BvT, bv)) ||
                (rc = dev_alloc(&s->ens_BvTs, 2 * bv)) || (rc = dev_alloc(&s->ens_BvTh, 2 * bv))) {
                set_error("out of device memory for the batched ensemble buffers (%d heads x %lld atoms)", HB, (long long)s->N);
                return rc;
            }
            s->ens_cap = HB;
        }
        if (HB >= 2 && pairbuf && (!s->ens_gbuf || s->ens_gcap < s->cap || s->ens_gheads < HB)) {  // heads' pair buffers
            dev_free(s->ens_gbuf); dev_free(s->ens_f);
            s->ens_gcap = 0, s->ens_gheads = 0;
            if ((rc = dev_alloc(&s->ens_gbuf, (size_t)s->N * s->cap * HB)) || (rc = dev_alloc(&s->ens_f, (size_t)3 * s->N * HB))) {
                set_error("out of device memory for the batched pair buffers (%d heads x %lld atoms x %d)", HB, (long long)s->N, s->cap);
                return rc;
            }
            s->ens_gcap = s->cap, s->ens_gheads = HB;
        }
    }
    const bool heads_kernel = HB >= 2 && s->force_mode == GMNN_FORCE_PAIRBUF && s->list_has_rev && s->ens_gbuf;
    struct BatchOff {  // the batch state never outlives the pass
        gmnn_system *s;
        ~BatchOff() { s->ens_batch = 0, s->ens_head = 0; }
    } batch_off{s};
    for (int m0 = 0; m0 < M; m0 += HB) {
        const int hb = std::min(HB, M - m0);
        if (s->mlp_precision == GMNN_MLP_3XF16 && m0 > 0)  // dZ maxima belong to one backward pass
            GMNN_CUDA(cudaMemsetAsync(s->amax + AMAX_DZ, 0, sizeof(uint32_t) * 2, st));
        if (HB >= 2) {
            if ((rc = launch_mlp_backward_tc_heads(s, m0, hb, st))) return rc;
            s->ens_batch = hb;
            if ((rc = launch_contract_backward(s, st))) return rc;
        }
        if (heads_kernel) {  // pair backward of the whole batch: geometry and radial functions once per pair and head chunk
            if ((rc = launch_pair_backward_heads_welford(s, m0, hb, f_mean, f_var, st))) return rc;
            s->ens_batch = 0;
            continue;
        }
        for (int mm = 0; mm < hb; ++mm) {
            const int m = m0 + mm;
            if (HB >= 2) {
                s->ens_head = mm;
            } else {
                k_set_onehot<<<1, 64, 0, st>>>(M, m, s->head_w);
                GMNN_LAUNCHED();
                if ((rc = mlp_backward(s, s->head_w, st))) return rc;
                if ((rc = launch_contract_backward(s, st))) return rc;
            }
            // pair backward of head m; its force goes straight into the statistics over the heads (no scatter, no store)
            if ((rc = launch_pair_backward_welford(s, m, f_mean, f_var, st))) return rc;
        }
        s->ens_batch = 0;
    }
    if ((rc = launch_finish_var(3 * s->N, f_var, M, st))) return rc;
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

}  // namespace gmnn

using namespace gmnn;

extern "C" {

const char *gmnn_last_error(void) { return g_error; }
int64_t gmnn_launch_count(void) { return (int64_t)g_launch_count; }

int32_t gmnn_n_features(int32_t n) {
    const int p = n * (n + 1) / 2, t = n * (n + 1) * (n + 2) / 6;
    return n + 3 * p + t + 2 * p * n + n * n * n;
}

int gmnn_create(const gmnn_hparams *hp, const gmnn_weights *w, gmnn_model **out) {
    if (!hp || !w || !out) {
        set_error("gmnn_create: null argument");
        return GMNN_INVALID_ARG;
    }
    if (hp->l_max != 3) {
        set_error("l_max must be 3 (got %d)", hp->l_max);
        return GMNN_UNSUPPORTED;
    }
    if (hp->n_species < 1 || hp->n_species > MAX_SPECIES || hp->n_basis < 2 || hp->n_basis > MAX_BASIS ||
        hp->n_radial < 1 || hp->n_hidden < 1 || hp->n_hidden > 4 || hp->n_heads < 1 || hp->n_heads > 64 ||
        !(hp->r_cut > 0.f) || !(hp->r_min >= 0.f) || !(hp->r_min < hp->r_cut) || !std::isfinite(hp->r_cut)) {
        set_error("gmnn_create: hyper-parameter out of range");
        return GMNN_INVALID_ARG;
    }
    if (hp->n_radial != 5 || hp->n_basis != 7) {
        set_error("kernels are instantiated for n_radial = 5, n_basis = 7 (got %d, %d)", hp->n_radial, hp->n_basis);
        return GMNN_UNSUPPORTED;
    }
    if (hp->radial_basis != 0 && hp->radial_basis != 1) {
        set_error("radial_basis must be 0 (Gaussians) or 1 (Bessel-like)");
        return GMNN_INVALID_ARG;
    }
    if (hp->zbl != 0) {
        if (!w->atomic_numbers || !(hp->zbl_r_max > 0.f) || !(hp->zbl_r_max <= hp->r_cut) || !std::isfinite(hp->zbl_scale)) {
            set_error("zbl needs atomic_numbers, 0 < zbl_r_max <= r_cut and a finite zbl_scale");
            return GMNN_INVALID_ARG;
        }
        for (int z = 0; z < hp->n_species; ++z)
            if (!(w->atomic_numbers[z] >= 1.f) || !(w->atomic_numbers[z] <= 120.f)) {
                set_error("atomic_numbers[%d] = %g is not a nuclear charge", z, w->atomic_numbers[z]);
                return GMNN_INVALID_ARG;
            }
    }
    if (hp->n_weight_sets != 1 && hp->n_weight_sets != hp->n_species) {
        set_error("n_weight_sets = %d: must be 1 (one NN for all species) or n_species = %d (one NN per species)",
                  hp->n_weight_sets, hp->n_species);
        return GMNN_INVALID_ARG;
    }
    if (hp->mlp_precision < 0 || hp->mlp_precision > GMNN_MLP_3XF16 || hp->force_mode < 0 ||
        hp->force_mode > GMNN_FORCE_PAIRBUF) {
        set_error("gmnn_create: bad mlp_precision / force_mode");
        return GMNN_INVALID_ARG;
    }
    for (int l = 0; l < hp->n_hidden; ++l)
        if (hp->hidden[l] < 16 || hp->hidden[l] > 1024 || hp->hidden[l] % 16 != 0) {
            set_error("hidden[%d] = %d must be a multiple of 16 in [16, 1024]", l, hp->hidden[l]);
            return GMNN_INVALID_ARG;
        }
    if (!w->beta || !w->scale || !w->shift) {
        set_error("gmnn_create: null weight pointer");
        return GMNN_INVALID_ARG;
    }
    for (int l = 0; l <= hp->n_hidden; ++l)
        if (!w->W[l] || !w->b[l]) {
            set_error("gmnn_create: null weight pointer (layer %d)", l);
            return GMNN_INVALID_ARG;
        }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        set_error("no CUDA device: this library has no CPU fallback");
        return GMNN_CUDA_ERROR;
    }
    gmnn_model *m = new gmnn_model();
    m->hp = *hp;
    cudaGetDevice(&m->device);
    m->n_features = gmnn_n_features(hp->n_radial);
    m->n_layers = hp->n_hidden + 1;
    m->dims[0] = m->n_features;
    for (int l = 0; l < hp->n_hidden; ++l) m->dims[l + 1] = hp->hidden[l];
    m->dims[hp->n_hidden + 1] = hp->n_heads;
    RadialParams &rp = m->rp;
    rp.n_species = hp->n_species;
    rp.n_basis = hp->n_basis;
    rp.kb = (hp->n_basis + 3) & ~3;
    rp.r_cut = hp->r_cut;
    rp.r_cut2 = hp->r_cut * hp->r_cut;
    rp.inv_rc = 1.f / hp->r_cut;
    rp.r_min = hp->r_min;
    rp.delta = (hp->r_cut - hp->r_min) / (float)(hp->n_basis - 1);
    rp.gamma = hp->gauss_gamma > 0.f ? hp->gauss_gamma : 1.f / (2.f * rp.delta * rp.delta);
    rp.basis_kind = hp->radial_basis;
    for (int n = 0; n < hp->n_basis; ++n)
        rp.bessel_c[n] = (float)(((n & 1) ? -1.0 : 1.0) * std::sqrt(2.0) * M_PI / std::pow((double)hp->r_cut, 1.5) * (n + 1.0) *
                                 (n + 2.0) / std::sqrt((n + 1.0) * (n + 1.0) + (n + 2.0) * (n + 2.0)));
    rp.zbl_on = hp->zbl != 0;
    if (rp.zbl_on) {
        rp.zbl_r_max2 = hp->zbl_r_max * hp->zbl_r_max;
        rp.zbl_inv_rmax = 1.f / hp->zbl_r_max;
        rp.zbl_pref = (float)(0.5 * (double)hp->zbl_scale * 14.399645);
        for (int z = 0; z < hp->n_species; ++z) {
            rp.zbl_z[z] = w->atomic_numbers[z];
            rp.zbl_zpow[z] = (float)std::pow((double)w->atomic_numbers[z], 0.23);
        }
    }
    int rc = GMNN_OK;
    {
        const int S = hp->n_species, nr = hp->n_radial, nb = hp->n_basis;
        std::vector<float> padded((size_t)S * S * nr * rp.kb, 0.f);
        for (int p = 0; p < S * S; ++p)
            for (int s = 0; s < nr; ++s)
                for (int k = 0; k < nb; ++k) padded[((size_t)p * nr + s) * rp.kb + k] = w->beta[((size_t)p * nr + s) * nb + k];
        rc = upload(&m->beta, padded.data(), padded.size());
    }
    const int T = m->n_sets = hp->n_weight_sets;
    for (int l = 0; l < m->n_layers && !rc; ++l) {
        const int fi = m->dims[l], fo = m->dims[l + 1];
        const size_t ws = (size_t)fi * fo;  // one set
        rc = upload(&m->W[l], w->W[l], ws * T);
        if (!rc) rc = upload(&m->b[l], w->b[l], (size_t)fo * T);
        std::vector<float> t(ws * T);
        for (int q = 0; q < T; ++q)
            for (int a = 0; a < fi; ++a)
                for (int b = 0; b < fo; ++b) t[q * ws + (size_t)b * fi + a] = w->W[l][q * ws + (size_t)a * fo + b];
        if (!rc) rc = upload(&m->WT[l], t.data(), t.size());
        if (!rc) rc = dev_alloc(&m->Ws[l], 2 * ws * T);
        if (!rc) rc = dev_alloc(&m->WTs[l], 2 * ws * T);
        if (!rc && l == 0) rc = dev_alloc(&m->wmax, (size_t)MAX_LAYERS);
        if (!rc) rc = dev_alloc(&m->Wh[l], 2 * ws * T);
        if (!rc) rc = dev_alloc(&m->WTh[l], 2 * ws * T);
        // one fp16 scale per layer, from the maximum over all of its sets
        if (!rc) rc = launch_absmax(m->W[l], (int64_t)(ws * T), m->wmax + l, nullptr);
        for (int q = 0; q < T && !rc; ++q) {
            rc = launch_split_stack(m->W[l] + q * ws, m->Ws[l] + 2 * q * ws, (int64_t)ws, nullptr);
            if (!rc) rc = launch_split_stack(m->WT[l] + q * ws, m->WTs[l] + 2 * q * ws, (int64_t)ws, nullptr);
            if (!rc) rc = launch_split_stack_h(m->W[l] + q * ws, m->Wh[l] + 2 * q * ws, (int64_t)ws, m->wmax + l, nullptr);
            if (!rc) rc = launch_split_stack_h(m->WT[l] + q * ws, m->WTh[l] + 2 * q * ws, (int64_t)ws, m->wmax + l, nullptr);
        }
    }
    if (!rc && cudaDeviceSynchronize() != cudaSuccess) rc = GMNN_CUDA_ERROR;
    if (!rc) rc = upload(&m->scale, w->scale, (size_t)hp->n_species);
    if (!rc) rc = upload(&m->shift, w->shift, (size_t)hp->n_species);
    if (!rc) {
        std::vector<float> hw(hp->n_heads, 1.f / (float)hp->n_heads);
        rc = upload(&m->head_mean_w, hw.data(), hw.size());
    }
    if (!rc) {
        // the mean of the heads is itself one linear head (Eq. 6, left-hand side): w_mean = W_last 1/M, b_mean
        const int L = hp->n_hidden, Hd = m->dims[L], M = hp->n_heads;
        std::vector<float> wm(((size_t)Hd + 1) * T);
        for (int q = 0; q < T; ++q)
            for (int k = 0; k <= Hd; ++k) {
                const float *row = (k < Hd) ? w->W[L] + ((size_t)q * Hd + k) * M : w->b[L] + (size_t)q * M;
                double acc = 0.0;
                for (int j = 0; j < M; ++j) acc += (double)row[j];
                wm[(size_t)q * (Hd + 1) + k] = (float)(acc / M);
            }
        rc = upload(&m->w_mean, wm.data(), wm.size());
    }
    if (rc) {
        gmnn_destroy(m);
        return rc;
    }
    *out = m;
    return GMNN_OK;
}

void gmnn_destroy(gmnn_model *m) {
    if (!m) return;
    dev_free(m->beta);
    dev_free(m->w_mean);
    for (int l = 0; l < MAX_LAYERS; ++l) {
        dev_free(m->W[l]);
        dev_free(m->WT[l]);
        dev_free(m->Ws[l]);
        dev_free(m->WTs[l]);
        dev_free(m->Wh[l]);
        dev_free(m->WTh[l]);
        dev_free(m->b[l]);
    }
    dev_free(m->scale);
    dev_free(m->shift);
    dev_free(m->head_mean_w);
    dev_free(m->wmax);
    delete m;
}

int gmnn_system_create(const gmnn_model *m, int64_t n_atoms, const int32_t *species, gmnn_system **out) {
    if (!m || !species || !out || n_atoms <= 0) {
        set_error("gmnn_system_create: null argument or n_atoms <= 0");
        return GMNN_INVALID_ARG;
    }
    if (n_atoms >= MAX_ATOMS) {
        set_error("n_atoms = %lld exceeds the %lld the packed neighbour entries can address", (long long)n_atoms,
                  (long long)MAX_ATOMS);
        return GMNN_UNSUPPORTED;
    }
    for (int64_t i = 0; i < n_atoms; ++i)
        if (species[i] < 0 || species[i] >= m->hp.n_species) {
            set_error("species[%lld] = %d out of range", (long long)i, species[i]);
            return GMNN_INVALID_ARG;
        }
    if (int rcd = check_device(m->device, "gmnn_system_create")) return rcd;
    gmnn_system *s = new gmnn_system();
    s->model = m;
    s->device = m->device;
    s->N = n_atoms;
    s->mlp_precision = m->hp.mlp_precision;
    s->force_mode = m->hp.force_mode;
    const size_t N = (size_t)n_atoms;
    const int F = m->n_features, L = m->hp.n_hidden, M = m->hp.n_heads;
    const int T = m->n_sets;
    int maxw = 0;
    for (int l = 1; l <= L; ++l) maxw = std::max(maxw, m->dims[l]);
    // rows of the MLP stage: atom order with one weight set, species segments padded to 256 rows otherwise
    s->n_rows = n_atoms;
    if (T > 1) {
        int64_t cnt[MAX_SPECIES] = {}, row = 0;
        for (size_t i = 0; i < N; ++i) cnt[species[i]]++;
        for (int z = 0; z < m->hp.n_species; ++z) {
            s->seg_row0[z] = row;
            s->seg_rows[z] = cnt[z];
            row += (cnt[z] + 255) / 256 * 256;
        }
        s->n_rows = row;
    }
    const size_t R = (size_t)s->n_rows;
    int rc = upload(&s->species, species, N);
#define A_(p, n) if (!rc) rc = dev_alloc(&(p), (n))
    A_(s->cell_of, N);
    A_(s->slot_tmp, N);
    A_(s->perm, N);
    A_(s->pos4, N);
    A_(s->xref, 3 * N);
    A_(s->count, N);
    A_(s->psi, R * m->hp.n_radial * PSI);
    // every matrix of the MLP is tile-transposed, [rows/128][width][128], padded to whole tiles (mlp_tc.cu)
    const size_t NP = (size_t)((R + 127) / 128 * 128);
    A_(s->G, NP * F);
    A_(s->dG, NP * F);
    A_(s->A, R * m->hp.n_radial * PSI);
    for (int l = 0; l < L; ++l) {
        A_(s->H[l], NP * m->dims[l + 1]);
        A_(s->D[l], NP * m->dims[l + 1]);
    }
    A_(s->dZ[0], NP * maxw);
    A_(s->dZ[1], NP * maxw);
    const size_t bv = (size_t)m->dims[L] * m->dims[L - 1];  // per weight set
    A_(s->Bv, bv * T);
    A_(s->BvT, bv * T);
    A_(s->BvTs, 2 * bv * T);
    A_(s->BvTh, 2 * bv * T);
    A_(s->amax, (size_t)AMAX_SLOTS);
    A_(s->vhead, (size_t)m->dims[L] * T);
    A_(s->head_w, (size_t)M);
    A_(s->ypart, (size_t)MAX_HEAD_SLOTS * NP);
    A_(s->e_heads, N * M);
    A_(s->e_atom, N);
    A_(s->f_int, 3 * N);
    A_(s->f_tmp, 3 * N);
    A_(s->partial, 2 * 1024);
    A_(s->e_total, 6);  // epot, ekin, sigma_E, bits of sigma_F,max (switching-mode samples)
    A_(s->flags, FLAG_WORDS);
    if (m->rp.zbl_on) A_(s->e_zbl, N);
    if (T > 1) {
        A_(s->mrow, N);
        A_(s->row_atom, R);
        A_(s->sp_count, ((N + 255) / 256 + 1) * MAX_SPECIES);
    }
#undef A_
    if (!rc && cudaMallocHost((void **)&s->flags_host, sizeof(int32_t) * FLAG_WORDS) != cudaSuccess) rc = GMNN_OOM;
    if (!rc && cudaMemset(s->flags, 0, sizeof(int32_t) * FLAG_WORDS) != cudaSuccess) rc = GMNN_CUDA_ERROR;
    if (!rc && cudaMemset(s->G, 0, sizeof(float) * NP * F) != cudaSuccess) rc = GMNN_CUDA_ERROR;  // rows of the ragged last tile
    if (!rc && T > 1) {  // padding rows: no moments (so G = 0 there), no atom
        if (cudaMemset(s->psi, 0, sizeof(float) * R * m->hp.n_radial * PSI) != cudaSuccess) rc = GMNN_CUDA_ERROR;
        if (!rc && cudaMemset(s->row_atom, 0xFF, sizeof(int32_t) * R) != cudaSuccess) rc = GMNN_CUDA_ERROR;
    }
    if (!rc && cudaMemset(s->amax, 0, sizeof(uint32_t) * AMAX_SLOTS) != cudaSuccess) rc = GMNN_CUDA_ERROR;
    if (!rc) {  // swish' lies in [-0.1, 1.1]: its scale is a constant
        const float dmax = 1.5f;
        if (cudaMemcpy(s->amax + AMAX_D, &dmax, sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) rc = GMNN_CUDA_ERROR;
    }
    if (rc) {
        if (rc == GMNN_OOM) set_error("out of device memory allocating the workspaces of %lld atoms", (long long)n_atoms);
        gmnn_system_destroy(s);
        return rc;
    }
    *out = s;
    return GMNN_OK;
}

void gmnn_system_destroy(gmnn_system *s) {
    if (!s) return;
    if (s->ef_exec) cudaGraphExecDestroy(s->ef_exec);
    dev_free(s->mrow); dev_free(s->row_atom); dev_free(s->sp_count); dev_free(s->vir_atom); dev_free(s->e_zbl);
    dev_free(s->species); dev_free(s->cell_of); dev_free(s->cell_count); dev_free(s->cell_start);
    dev_free(s->cell_fill); dev_free(s->slot_tmp); dev_free(s->perm); dev_free(s->pos4); dev_free(s->xref);
    dev_free(s->nbr); dev_free(s->rev); dev_free(s->gbuf); dev_free(s->runs); dev_free(s->count); dev_free(s->psi); dev_free(s->G); dev_free(s->dG); dev_free(s->A);
    for (int l = 0; l < MAX_LAYERS; ++l) { dev_free(s->H[l]); dev_free(s->D[l]); }
    dev_free(s->dZ[0]); dev_free(s->dZ[1]); dev_free(s->Bv); dev_free(s->BvT); dev_free(s->BvTs); dev_free(s->BvTh); dev_free(s->amax); dev_free(s->vhead); dev_free(s->head_w);
    dev_free(s->ypart); dev_free(s->e_heads); dev_free(s->e_atom); dev_free(s->f_int); dev_free(s->f_tmp); dev_free(s->partial);
    dev_free(s->e_total); dev_free(s->flags); dev_free(s->ens_scratch); dev_free(s->nhc); dev_free(s->lang_step);
    dev_free(s->ens_dZ[0]); dev_free(s->ens_dZ[1]); dev_free(s->ens_dG); dev_free(s->ens_A); dev_free(s->ens_gbuf); dev_free(s->ens_f);
    dev_free(s->ens_BvT); dev_free(s->ens_BvTs); dev_free(s->ens_BvTh);
    dev_free(s->kT_now); dev_free(s->sched_steps); dev_free(s->sched_temps); dev_free(s->sched_step);
    dev_free(s->stage_pos); dev_free(s->stage_f); dev_free(s->stage_e);
    if (s->flags_host) cudaFreeHost(s->flags_host);
    for (cudaEvent_t e : s->events) cudaEventDestroy(e);
    if (s->graph_stream) {
        cudaStreamDestroy(s->graph_stream);
        cudaEventDestroy(s->graph_ev[0]);
        cudaEventDestroy(s->graph_ev[1]);
    }
    delete s;
}

int gmnn_system_set_int(gmnn_system *s, const char *key, int64_t v) {
    if (!s || !key) return GMNN_INVALID_ARG;
    ++g_config_gen;  // any knob may change what an evaluation launches
    s->seed_w = nullptr;
    if (!strcmp(key, "lanes_per_atom")) {
        if (v != 0 && v != 1 && v != 2 && v != 4 && v != 8 && v != 16 && v != 32) {
            set_error("lanes_per_atom must be 0, 1, 2, 4, 8, 16 or 32");
            return GMNN_INVALID_ARG;
        }
        s->lanes_per_atom = (int)v;
    } else if (!strcmp(key, "profile")) {
        s->profile = v != 0;
        s->n_stage_events = 0;
        // events are created here, not lazily inside the calls being timed (a few microseconds each, 13 per MD step)
        while (s->profile && s->events.size() < 2048) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) break;
            s->events.push_back(e);
            s->stage_names.push_back(nullptr);
        }
    } else if (!strcmp(key, "ensemble_batch")) {
        if (v < 0 || v > 64) {
            set_error("ensemble_batch must be in [0, 64]");
            return GMNN_INVALID_ARG;
        }
        s->ens_batch_max = (int)v;
    } else if (!strcmp(key, "md_continue")) {
        s->md_continue = v != 0;
    } else if (!strcmp(key, "md_graph")) {
        s->md_graph = v != 0;
    } else if (!strcmp(key, "ef_graph")) {
        s->ef_graph = v != 0;
    } else if (!strcmp(key, "capacity")) {
        if (v < 0 || v > 4096) {
            set_error("capacity must be in [0, 4096]");
            return GMNN_INVALID_ARG;
        }
        s->cap_request = (int)v;
    } else if (!strcmp(key, "mlp_precision")) {
        if (v < 0 || v > GMNN_MLP_3XF16) return GMNN_INVALID_ARG;
        s->mlp_precision = (int)v;
    } else if (!strcmp(key, "force_mode")) {
        if (v < 0 || v > GMNN_FORCE_PAIRBUF) return GMNN_INVALID_ARG;
        if (s->force_mode != (int)v) s->have_list = false;  // the reverse-pair index is built with the list
        s->force_mode = (int)v;
    } else if (!strcmp(key, "tc_split_bk")) {  // process-wide tuning knob of mlp_tc.cu
        if (v != 16 && v != 32) return GMNN_INVALID_ARG;
        gmnn::g_tc_split_bk = (int)v;
#ifdef GMNN_EXPERIMENTS
    } else if (!strcmp(key, "cb_halves")) {  // superseded block shapes of k_contract_backward (descriptor.cu)
        if (v < 1 || v > 6) return GMNN_INVALID_ARG;
        gmnn::g_cb_halves = (int)v;
    } else if (!strcmp(key, "tc_debug")) {  // knock-out timing experiments (wrong results), see mlp_tc.cu
        gmnn::g_tc_debug = (int)v;
#endif
    } else if (!strcmp(key, "tc_fwd_scheme")) {  // process-wide, see mlp_tc.cu
        if (v < 1 || v > 2) return GMNN_INVALID_ARG;
        gmnn::g_tc_fwd_scheme = (int)v;
    } else if (!strcmp(key, "tc_tile_order")) {  // process-wide, see mlp_tc.cu
        if (v < 0 || v > 3) return GMNN_INVALID_ARG;
        gmnn::g_tc_tile_order = (int)v;
    } else if (!strcmp(key, "tc_dmul_prefetch")) {  // process-wide, see mlp_tc.cu
        if (v < -1 || v > 64) return GMNN_INVALID_ARG;
        gmnn::g_tc_dmul_prefetch = (int)v;
    } else if (!strcmp(key, "tc_flush_k_bwd")) {  // process-wide, see mlp_tc.cu
        if (v < 16 || v > 4096 || v % 16) return GMNN_INVALID_ARG;
        gmnn::g_tc_flush_k_bwd = (int)v;
    } else if (!strcmp(key, "tc_pair")) {  // process-wide: 3xTF32 GEMMs on CTA pairs (1) or single CTAs (0)
        gmnn::g_tc_pair = v != 0;
    } else if (!strcmp(key, "tc_h_bk")) {  // process-wide: K extent of a 3xFP16 stage
        if (v != 32 && v != 64) return GMNN_INVALID_ARG;
        gmnn::g_tc_h_bk = (int)v;
    } else if (!strcmp(key, "tc_flush_k")) {
        if (v < 16 || v > 4096 || v % 16) return GMNN_INVALID_ARG;
        gmnn::g_tc_flush_k = (int)v;
    } else {
        set_error("unknown key '%s'", key);
        return GMNN_INVALID_ARG;
    }
    return GMNN_OK;
}

int gmnn_system_get_int(const gmnn_system *s, const char *key, int64_t *v) {
    if (!s || !key || !v) return GMNN_INVALID_ARG;
    if (!strcmp(key, "lanes_per_atom")) *v = s->lanes_per_atom;
    else if (!strcmp(key, "ensemble_batch")) *v = s->ens_batch_max;
    else if (!strcmp(key, "profile")) *v = s->profile;
    else if (!strcmp(key, "md_continue")) *v = s->md_continue;
    else if (!strcmp(key, "md_graph")) *v = s->md_graph;
    else if (!strcmp(key, "ef_graph")) *v = s->ef_graph;
    else if (!strcmp(key, "capacity")) *v = s->cap;
    else if (!strcmp(key, "mlp_precision")) *v = s->mlp_precision;
    else if (!strcmp(key, "force_mode")) *v = s->force_mode;
    else if (!strcmp(key, "n_cells")) *v = s->ncells;
    else if (!strcmp(key, "small_box")) *v = s->small_box;
    else {
        set_error("unknown key '%s'", key);
        return GMNN_INVALID_ARG;
    }
    return GMNN_OK;
}

static int read_flags(gmnn_system *s, cudaStream_t st) {
    GMNN_CUDA(cudaMemcpyAsync(s->flags_host, s->flags, sizeof(int32_t) * FLAG_WORDS, cudaMemcpyDeviceToHost, st));
    GMNN_CUDA(cudaStreamSynchronize(st));
    return GMNN_OK;
}

int gmnn_build_neighbors(gmnn_system *s, const float *positions, const float cell[9], const int32_t pbc[3],
                         float r_cut, float skin, void *cuda_stream) {
    if (!s || !positions || !cell || !pbc) {
        set_error("gmnn_build_neighbors: null argument");
        return GMNN_INVALID_ARG;
    }
    if (int rcd = check_device(s->device, "gmnn_build_neighbors")) return rcd;
    ++g_config_gen;  // geometry, capacity and buffers may change
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (r_cut != s->model->hp.r_cut) {
        set_error("r_cut = %g differs from the model's %g", r_cut, s->model->hp.r_cut);
        return GMNN_INVALID_ARG;
    }
    if (!(skin >= 0.f) || !std::isfinite(skin)) {
        set_error("skin must be finite and >= 0");
        return GMNN_INVALID_ARG;
    }
    bool triclinic = false;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            const float v = cell[3 * a + b];
            if (!std::isfinite(v) || (a == b && !(v > 0.f))) {
                set_error("cell must be finite with positive diagonal");
                return GMNN_INVALID_ARG;
            }
            if (a != b && v != 0.f) triclinic = true;
        }
    // general lattice (rows a, b, c): volume, inverse and the distances w_a between opposite faces, in fp64
    double hd[9], hinv[9], w[3], cell_volume = 0.0;
    for (int q = 0; q < 9; ++q) hd[q] = (double)cell[q];
    {
        const double *a = hd, *b = hd + 3, *c = hd + 6;
        const double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
        const double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
        const double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
        const double det = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
        if (!(std::fabs(det) > 1e-6)) {
            set_error("cell is singular (volume %g)", det);
            return GMNN_INVALID_ARG;
        }
        cell_volume = std::fabs(det);
        w[0] = std::fabs(det) / std::sqrt(bc[0] * bc[0] + bc[1] * bc[1] + bc[2] * bc[2]);
        w[1] = std::fabs(det) / std::sqrt(ca[0] * ca[0] + ca[1] * ca[1] + ca[2] * ca[2]);
        w[2] = std::fabs(det) / std::sqrt(ab[0] * ab[0] + ab[1] * ab[1] + ab[2] * ab[2]);
        // x (row) . hinv = fractional coordinates: columns of hinv are the reciprocal vectors
        for (int x = 0; x < 3; ++x) hinv[3 * x + 0] = bc[x] / det, hinv[3 * x + 1] = ca[x] / det, hinv[3 * x + 2] = ab[x] / det;
    }
    s->md_state_valid = false;
    // The handle holds no usable list from here until this call succeeds: an earlier list must never
    // sit beside the new geometry, a freed row buffer or truncated rows (every failure path below
    // returns with have_list == false).  The new geometry is filled locally and committed once valid.
    s->have_list = false;
    Geometry g{};
    const float r_list = r_cut + skin;  // fl32(fl32(r_cut) + fl32(skin)): the oracle is handed the same float
    g.r_list2 = r_list * r_list;
    g.r_cut2 = r_cut * r_cut;
    g.triclinic = triclinic ? 1 : 0;
    for (int q = 0; q < 9; ++q) g.h[q] = cell[q], g.hinv[q] = (float)hinv[q];
    bool small = false;
    for (int a = 0; a < 3; ++a) {
        g.L[a] = cell[4 * a];
        g.invL[a] = 1.f / g.L[a];
        g.pbc[a] = pbc[a] != 0;
        // slabs at least r_list thick between the faces of axis a (w_a = L_a for an orthorhombic cell)
        const double width = triclinic ? w[a] : (double)g.L[a];
        int nc = (int)std::floor(width / ((double)r_list * (1.0 + 1e-5)));
        if (nc < 1) nc = 1;
        if (nc > 1024) nc = 1024;
        g.ncell[a] = nc;
        if (g.pbc[a] && nc < 3) small = true;
    }
    if (small) {
        if (s->N > SMALL_BOX_MAX_ATOMS) {
            set_error("box has < 3 cells on a periodic axis: the all-pairs image path is limited to %d atoms",
                      SMALL_BOX_MAX_ATOMS);
            return GMNN_UNSUPPORTED;
        }
        for (int a = 0; a < 3; ++a) {
            // orthorhombic: fp32 division, as the oracle's ceilf; general lattice: the face distance
            g.kimg[a] = !g.pbc[a] ? 0 : triclinic ? (int)std::ceil((double)r_list / w[a]) : (int)std::ceil(r_list / g.L[a]);
            if (g.kimg[a] > 3) {
                set_error("box needs more than 3 periodic images along axis %d at r_list = %g", a, r_list);
                return GMNN_UNSUPPORTED;
            }
            g.ncell[a] = 1;
        }
    } else {
        g.kimg[0] = g.kimg[1] = g.kimg[2] = 0;
    }
    for (int a = 0; a < 3; ++a) g.inv_edge[a] = (float)g.ncell[a] / g.L[a];
    s->geo = g;
    s->small_box = small;
    s->r_cut = r_cut;
    s->skin = skin;
    s->ncells = (int64_t)g.ncell[0] * g.ncell[1] * g.ncell[2];
    if (s->ncells > s->ncells_alloc) {
        dev_free(s->cell_count);
        dev_free(s->cell_start);
        dev_free(s->cell_fill);
        int rc = dev_alloc(&s->cell_count, (size_t)s->ncells + 1);
        if (!rc) rc = dev_alloc(&s->cell_start, (size_t)s->ncells + 1);
        if (!rc) rc = dev_alloc(&s->cell_fill, (size_t)s->ncells);
        if (rc) return rc;
        s->ncells_alloc = s->ncells;
    }
    // capacity: expected neighbours at uniform density x 1.3 + 32, a multiple of 32
    int want = s->cap_request;
    if (want <= 0) {
        const double per = (double)s->N / cell_volume * 4.0 / 3.0 * M_PI * std::pow((double)r_list, 3.0);
        want = (int)(per * 1.3) + 32;
    }
    want = (want + 31) & ~31;
    for (int attempt = 0; attempt < 4; ++attempt) {
        if (want > s->cap || !s->nbr) {
            dev_free(s->nbr);
            s->cap = want;
            int rc = dev_alloc(&s->nbr, (size_t)s->N * s->cap);
            dev_free(s->rev);
            dev_free(s->gbuf);
            if (rc) {
                set_error("out of device memory for the neighbour list (%lld x %d)", (long long)s->N, s->cap);
                s->cap = 0;
                return rc;
            }
        }
        if (s->force_mode == GMNN_FORCE_PAIRBUF && !s->rev) {
            int rc = dev_alloc(&s->rev, (size_t)s->N * s->cap);
            if (!rc) rc = dev_alloc(&s->gbuf, (size_t)s->N * s->cap);
            if (!rc && !s->runs) rc = dev_alloc(&s->runs, (size_t)s->N * 56);
            if (rc) {
                set_error("out of device memory for the pair buffer (%lld x %d)", (long long)s->N, s->cap);
                return rc;
            }
        }
        s->list_has_rev = s->force_mode == GMNN_FORCE_PAIRBUF;
        GMNN_CUDA(cudaMemsetAsync(s->flags, 0, sizeof(int32_t) * FLAG_WORDS, st));
        int rc = launch_build(s, positions, st, nullptr, 0.f, false, nullptr);
        if (rc) return rc;
        if ((rc = read_flags(s, st))) return rc;
        if (s->flags_host[FLAG_OUT_OF_BOX]) {
            set_error("a position is outside [0, L): wrap positions before gmnn_build_neighbors");
            return GMNN_OUT_OF_BOX;
        }
        if (s->flags_host[FLAG_MAXCOUNT] <= s->cap) {
            if (s->flags_host[FLAG_REV_MISSING]) {
                set_error("internal: the neighbour list is not symmetric (reverse pair missing)");
                return GMNN_CUDA_ERROR;
            }
            s->have_list = true;
            GMNN_CUDA(cudaMemsetAsync(s->flags, 0, sizeof(int32_t) * FLAG_WORDS, st));
            return GMNN_OK;
        }
        want = ((int)(s->flags_host[FLAG_MAXCOUNT] * 1.15) + 32 + 31) & ~31;
    }
    set_error("neighbour list kept overflowing");
    return GMNN_NEIGHBOR_OVERFLOW;
}

int gmnn_get_neighbors(gmnn_system *s, int64_t *n_pairs, int32_t *oi, int32_t *oj, int32_t *oimg) {
    if (!s || !n_pairs) return GMNN_INVALID_ARG;
    if (!s->have_list) {
        set_error("no neighbour list: call gmnn_build_neighbors first");
        return GMNN_INVALID_ARG;
    }
    const size_t N = (size_t)s->N;
    std::vector<int32_t> cnt(N), perm(N);
    GMNN_CUDA(cudaDeviceSynchronize());
    GMNN_CUDA(cudaMemcpy(cnt.data(), s->count, sizeof(int32_t) * N, cudaMemcpyDeviceToHost));
    GMNN_CUDA(cudaMemcpy(perm.data(), s->perm, sizeof(int32_t) * N, cudaMemcpyDeviceToHost));
    int64_t total = 0;
    for (size_t k = 0; k < N; ++k) total += cnt[k];
    *n_pairs = total;
    if (!oi && !oj && !oimg) return GMNN_OK;
    if (!oi || !oj || !oimg) return GMNN_INVALID_ARG;
    std::vector<uint32_t> nbr(N * (size_t)s->cap);
    GMNN_CUDA(cudaMemcpy(nbr.data(), s->nbr, sizeof(uint32_t) * nbr.size(), cudaMemcpyDeviceToHost));
    struct Row { int32_t i, j, n[3]; };
    std::vector<Row> rows;
    rows.reserve((size_t)total);
    for (size_t k = 0; k < N; ++k)
        for (int q = 0; q < cnt[k]; ++q) {
            const uint32_t e = nbr[k * (size_t)s->cap + q];
            Row r;
            r.i = perm[k];
            r.j = perm[e & NBR_J_MASK];
            r.n[0] = (int)((e >> NBR_J_BITS) & 7u) - 4;
            r.n[1] = (int)((e >> (NBR_J_BITS + 3)) & 7u) - 4;
            r.n[2] = (int)((e >> (NBR_J_BITS + 6)) & 7u) - 4;
            rows.push_back(r);
        }
    std::sort(rows.begin(), rows.end(), [](const Row &a, const Row &b) {
        if (a.i != b.i) return a.i < b.i;
        if (a.j != b.j) return a.j < b.j;
        if (a.n[0] != b.n[0]) return a.n[0] < b.n[0];
        if (a.n[1] != b.n[1]) return a.n[1] < b.n[1];
        return a.n[2] < b.n[2];
    });
    for (size_t p = 0; p < rows.size(); ++p) {
        oi[p] = rows[p].i;
        oj[p] = rows[p].j;
        oimg[3 * p] = rows[p].n[0];
        oimg[3 * p + 1] = rows[p].n[1];
        oimg[3 * p + 2] = rows[p].n[2];
    }
    return GMNN_OK;
}

int gmnn_get_neighbor_rows(gmnn_system *s, int64_t n_sel, const int32_t *atoms, int64_t *n_pairs, int32_t *oi, int32_t *oj,
                           int32_t *oimg) {
    if (!s || !n_pairs || !atoms || n_sel < 0) return GMNN_INVALID_ARG;
    if (!s->have_list) {
        set_error("no neighbour list: call gmnn_build_neighbors first");
        return GMNN_INVALID_ARG;
    }
    const size_t N = (size_t)s->N;
    std::vector<int32_t> perm(N), inv(N);
    GMNN_CUDA(cudaDeviceSynchronize());
    GMNN_CUDA(cudaMemcpy(perm.data(), s->perm, sizeof(int32_t) * N, cudaMemcpyDeviceToHost));
    for (size_t k = 0; k < N; ++k) inv[perm[k]] = (int32_t)k;
    struct Row { int32_t i, j, n[3]; };
    std::vector<Row> rows;
    std::vector<uint32_t> buf((size_t)s->cap);
    for (int64_t q = 0; q < n_sel; ++q) {
        if (atoms[q] < 0 || (size_t)atoms[q] >= N) {
            set_error("gmnn_get_neighbor_rows: atom index %d out of range", atoms[q]);
            return GMNN_INVALID_ARG;
        }
        const size_t k = (size_t)inv[atoms[q]];
        int32_t cnt = 0;
        GMNN_CUDA(cudaMemcpy(&cnt, s->count + k, sizeof(int32_t), cudaMemcpyDeviceToHost));
        GMNN_CUDA(cudaMemcpy(buf.data(), s->nbr + k * (size_t)s->cap, sizeof(uint32_t) * (size_t)cnt, cudaMemcpyDeviceToHost));
        for (int c = 0; c < cnt; ++c) {
            const uint32_t e = buf[c];
            Row r;
            r.i = atoms[q];
            r.j = perm[e & NBR_J_MASK];
            r.n[0] = (int)((e >> NBR_J_BITS) & 7u) - 4;
            r.n[1] = (int)((e >> (NBR_J_BITS + 3)) & 7u) - 4;
            r.n[2] = (int)((e >> (NBR_J_BITS + 6)) & 7u) - 4;
            rows.push_back(r);
        }
    }
    *n_pairs = (int64_t)rows.size();
    if (!oi && !oj && !oimg) return GMNN_OK;
    if (!oi || !oj || !oimg) return GMNN_INVALID_ARG;
    std::stable_sort(rows.begin(), rows.end(), [](const Row &a, const Row &b) {
        if (a.i != b.i) return a.i < b.i;
        if (a.j != b.j) return a.j < b.j;
        if (a.n[0] != b.n[0]) return a.n[0] < b.n[0];
        if (a.n[1] != b.n[1]) return a.n[1] < b.n[1];
        return a.n[2] < b.n[2];
    });
    for (size_t p = 0; p < rows.size(); ++p) {
        oi[p] = rows[p].i;
        oj[p] = rows[p].j;
        oimg[3 * p] = rows[p].n[0];
        oimg[3 * p + 1] = rows[p].n[1];
        oimg[3 * p + 2] = rows[p].n[2];
    }
    return GMNN_OK;
}

int gmnn_energy_forces(gmnn_system *s, const float *positions, double *energy, float *energy_per_atom, float *forces,
                       void *cuda_stream) {
    if (!s || !positions || !energy || !forces) {
        set_error("gmnn_energy_forces: null argument");
        return GMNN_INVALID_ARG;
    }
    if (int rcd = check_device(s->device, "gmnn_energy_forces")) return rcd;
    if (!s->have_list) {
        set_error("no neighbour list: call gmnn_build_neighbors first");
        return GMNN_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->md_state_valid = false;
    StageTimer T(s, st);
    T.begin();
    int rc = forward_backward(s, positions, s->model->head_mean_w, true, st, T, true);
    if (rc) return rc;
    if ((rc = launch_scatter_outputs(s, energy_per_atom, forces, st))) return rc;
    if ((rc = launch_energy_sum(s, energy, st))) return rc;
    T.mark("outputs");
    return GMNN_OK;
}

int gmnn_energy_forces_virial(gmnn_system *s, const float *positions, double *energy, float *energy_per_atom,
                              float *forces, double *virial, void *cuda_stream) {
    if (!s || !virial) {
        set_error("gmnn_energy_forces_virial: null argument");
        return GMNN_INVALID_ARG;
    }
    if (!s->vir_atom) {  // per-atom virial terms [9][N], allocated at the first call that asks for the virial
        int rc = dev_alloc(&s->vir_atom, (size_t)9 * (size_t)s->N);
        if (rc) return rc;
    }
    struct Want {
        gmnn_system *s;
        ~Want() { s->want_virial = false; }
    } guard{s};
    s->want_virial = true;
    int rc = gmnn_energy_forces(s, positions, energy, energy_per_atom, forces, cuda_stream);
    if (rc) return rc;
    return launch_virial_sum(s, virial, (cudaStream_t)cuda_stream);
}

int gmnn_energy_forces_host(gmnn_system *s, const float *positions, double *energy, float *energy_per_atom,
                            float *forces, void *cuda_stream) {
    if (!s || !positions || !energy || !forces) {
        set_error("gmnn_energy_forces_host: null argument");
        return GMNN_INVALID_ARG;
    }
    if (int rcd = check_device(s->device, "gmnn_energy_forces_host")) return rcd;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t N = (size_t)s->N;
    int rc = GMNN_OK;
    if (!s->stage_pos) {
        rc = dev_alloc(&s->stage_pos, 3 * N);
        if (!rc) rc = dev_alloc(&s->stage_f, 3 * N);
        if (!rc) rc = dev_alloc(&s->stage_e, N);
        if (rc) return rc;
    }
    GMNN_CUDA(cudaMemcpyAsync(s->stage_pos, positions, sizeof(float) * 3 * N, cudaMemcpyHostToDevice, st));
    rc = gmnn_energy_forces(s, s->stage_pos, s->e_total, energy_per_atom ? s->stage_e : nullptr, s->stage_f, st);
    if (rc) return rc;
    GMNN_CUDA(cudaMemcpyAsync(forces, s->stage_f, sizeof(float) * 3 * N, cudaMemcpyDeviceToHost, st));
    if (energy_per_atom)
        GMNN_CUDA(cudaMemcpyAsync(energy_per_atom, s->stage_e, sizeof(float) * N, cudaMemcpyDeviceToHost, st));
    GMNN_CUDA(cudaMemcpyAsync(energy, s->e_total, sizeof(double), cudaMemcpyDeviceToHost, st));
    GMNN_CUDA(cudaStreamSynchronize(st));
    return GMNN_OK;
}

int gmnn_ensemble_energy_forces(gmnn_system *s, const float *positions, float *e_mean, float *e_var, float *f_mean,
                                float *f_var, void *cuda_stream) {
    if (!s || !positions || !e_mean || !e_var || !f_mean || !f_var) {
        set_error("gmnn_ensemble_energy_forces: null argument");
        return GMNN_INVALID_ARG;
    }
    if (int rcd = check_device(s->device, "gmnn_ensemble_energy_forces")) return rcd;
    if (!s->have_list) {
        set_error("no neighbour list: call gmnn_build_neighbors first");
        return GMNN_INVALID_ARG;
    }
    s->md_state_valid = false;
    return ensemble_pass(s, positions, e_mean, e_var, f_mean, f_var, (cudaStream_t)cuda_stream);
}

int gmnn_md_verlet_steps(gmnn_system *s, float *positions, float *velocities, const float *masses, float dt_fs,
                         int32_t n_steps, double *epot_series, double *ekin_series, int32_t *n_rebuilds,
                         void *cuda_stream) {
    if (!s || !positions || !velocities || !masses || n_steps < 0 || !(dt_fs > 0.f)) {
        set_error("gmnn_md_verlet_steps: bad argument");
        return GMNN_INVALID_ARG;
    }
    if (int rcd = check_device(s->device, "gmnn_md_verlet_steps")) return rcd;
    if (!s->have_list) {
        set_error("no neighbour list: call gmnn_build_neighbors first");
        return GMNN_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const float hs = 0.5f * s->skin;
    const float thr2 = hs * hs;
    int rc;
    StageTimer T(s, st);
    T.begin();
    // several heads: the integrated energy is their mean, evaluated as ONE folded head (model->w_mean) so that
    // a step costs what it costs on a single-head model; e_heads is not produced in the loop
    struct MeanHead {
        gmnn_system *s;
        ~MeanHead() { s->use_mean_head = false; }
    } mean_head_guard{s};
    s->use_mean_head = s->model->hp.n_heads > 1;
    double *const ep = s->e_total, *const ek = s->e_total + 1;  // energies of the latest step (device)
    if (s->md_continue && s->md_state_valid) {
        // the caller continues the trajectory of the previous call: f_tmp, e_total are current
        if (epot_series) GMNN_CUDA(cudaMemcpyAsync(epot_series, ep, sizeof(double), cudaMemcpyDeviceToDevice, st));
        if (ekin_series) GMNN_CUDA(cudaMemcpyAsync(ekin_series, ek, sizeof(double), cudaMemcpyDeviceToDevice, st));
    } else {
        // state at entry: forces of the current positions; the skin test against the list's build positions
        // runs here too (a caller whose atoms moved > skin/2 since gmnn_build_neighbors gets
        // GMNN_STALE_NEIGHBORS at the end of this call instead of a silently stale first step)
        if ((rc = forward_backward(s, positions, s->model->head_mean_w, true, st, T))) return rc;
        if ((rc = launch_scatter_outputs(s, nullptr, s->f_tmp, st))) return rc;
        if ((rc = launch_energy_sum(s, ep, st, epot_series))) return rc;
        if ((rc = launch_ke(s, velocities, masses, ek, st, ekin_series))) return rc;
        T.mark("outputs");
    }
    s->md_state_valid = false;
    // One step: every launch has the same arguments at every step (the energies go to the series
    // through a device-side counter), so the body can be captured once and replayed as a CUDA graph.
    auto md_step = [&](cudaStream_t q) -> int {
        int r;
        // temperature schedule: this step's target for whichever thermostat is set
        if (s->sched_n > 0 && (s->nhc_len > 0 || s->lang_on) && (r = launch_schedule_eval(s, q))) return r;
        // NVT: chain operator for dt/2 before and after the velocity-Verlet step
        if (s->nhc_len > 0 && (r = launch_nhc_half(s, velocities, ek, dt_fs, q))) return r;
        if (s->lang_on) {  // Langevin: B A O A in one pass (the closing B is the kick below)
            if ((r = launch_baoab(s, positions, velocities, s->f_tmp, masses, dt_fs, q))) return r;
        } else if ((r = launch_kick_drift(s, positions, velocities, s->f_tmp, masses, dt_fs, q))) {
            return r;
        }
        T.mark("kick_drift");
        // rebuild (wrap first) iff the max displacement since the last build exceeds skin/2
        if ((r = launch_build(s, positions, q, s->flags + FLAG_DISP2, thr2, true, positions))) return r;
        T.mark("rebuild_if_moved");
        if ((r = forward_backward(s, positions, s->model->head_mean_w, false, q, T))) return r;
        if ((r = launch_scatter_outputs(s, nullptr, s->f_tmp, q))) return r;
        if ((r = launch_energy_sum(s, ep, q, nullptr))) return r;
        T.mark("outputs");
        if ((r = launch_kick_ke(s, velocities, s->f_tmp, masses, dt_fs, ek, q, nullptr))) return r;
        if (s->nhc_len > 0 && (r = launch_nhc_half(s, velocities, ek, dt_fs, q))) return r;
        if ((epot_series || ekin_series) && (r = launch_series_append(s, epot_series, ekin_series, q))) return r;
        T.mark("kick_ke");
        return GMNN_OK;
    };
    if (n_steps > 0 && (rc = launch_series_reset(s, 1, st))) return rc;
    int step = 1;
    // the first step runs eagerly (one-time function attributes and driver lookups happen there)
    if (n_steps >= 1) {
        if ((rc = md_step(st))) return rc;
        ++step;
    }
    if (step <= n_steps && s->md_graph && !s->profile && n_steps >= 4) {
        if (!s->graph_stream) {
            GMNN_CUDA(cudaStreamCreateWithFlags(&s->graph_stream, cudaStreamNonBlocking));
            GMNN_CUDA(cudaEventCreateWithFlags(&s->graph_ev[0], cudaEventDisableTiming));
            GMNN_CUDA(cudaEventCreateWithFlags(&s->graph_ev[1], cudaEventDisableTiming));
        }
        cudaStream_t q = s->graph_stream;
        GMNN_CUDA(cudaEventRecord(s->graph_ev[0], st));
        GMNN_CUDA(cudaStreamWaitEvent(q, s->graph_ev[0], 0));
        const long long launches_before = g_launch_count;
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        GMNN_CUDA(cudaStreamBeginCapture(q, cudaStreamCaptureModeThreadLocal));
        rc = md_step(q);
        const cudaError_t cap = cudaStreamEndCapture(q, &graph);
        if (rc || cap != cudaSuccess) {
            if (graph) cudaGraphDestroy(graph);
            if (!rc) {
                set_error("CUDA graph capture of the MD step failed: %s", cudaGetErrorString(cap));
                rc = GMNN_CUDA_ERROR;
            }
            return rc;
        }
        const long long per_step = g_launch_count - launches_before;  // captured, not yet run
        g_launch_count = launches_before;
        cudaError_t ge = cudaGraphInstantiate(&exec, graph, 0);
        for (; ge == cudaSuccess && step <= n_steps; ++step) {
            ge = cudaGraphLaunch(exec, q);
            g_launch_count += per_step;
        }
        if (exec) cudaGraphExecDestroy(exec);
        cudaGraphDestroy(graph);
        if (ge != cudaSuccess) {
            set_error("CUDA graph replay of the MD step failed: %s", cudaGetErrorString(ge));
            return GMNN_CUDA_ERROR;
        }
        GMNN_CUDA(cudaEventRecord(s->graph_ev[1], q));
        GMNN_CUDA(cudaStreamWaitEvent(st, s->graph_ev[1], 0));
    }
    for (; step <= n_steps; ++step)
        if ((rc = md_step(st))) return rc;
    if ((rc = read_flags(s, st))) return rc;
    if (n_rebuilds) *n_rebuilds = s->flags_host[FLAG_REBUILDS];
    const int maxcount = s->flags_host[FLAG_MAXCOUNT];
    const int rev_missing = s->flags_host[FLAG_REV_MISSING];
    const int stale = s->flags_host[FLAG_STALE], oob = s->flags_host[FLAG_OUT_OF_BOX];
    GMNN_CUDA(cudaMemsetAsync(s->flags, 0, sizeof(int32_t) * FLAG_WORDS, st));
    if (stale) {  // raised by the entry evaluation of this call or by an earlier gmnn_energy_forces
        set_error("an atom had moved more than skin/2 from the positions the neighbour list was built at when "
                  "gmnn_md_verlet_steps was entered: call gmnn_build_neighbors first");
        return GMNN_STALE_NEIGHBORS;
    }
    if (oob) {  // k_wrap folds periodic axes only: an atom left the box along a non-periodic axis
        set_error("an atom left the box along a non-periodic axis at an in-loop rebuild (cells there clamp to the edge)");
        return GMNN_OUT_OF_BOX;
    }
    if (rev_missing && maxcount <= s->cap) {
        set_error("internal: an in-loop rebuild produced a neighbour list that is not symmetric");
        return GMNN_CUDA_ERROR;
    }
    if (maxcount > s->cap) {
        set_error("an in-loop rebuild needed %d neighbour slots, capacity is %d: raise \"capacity\" and rerun", maxcount,
                  s->cap);
        return GMNN_NEIGHBOR_OVERFLOW;
    }
    s->md_state_valid = true;
    return GMNN_OK;
}

int gmnn_md_ensemble_steps(gmnn_system *s, float *positions, float *velocities, const float *masses, float dt_fs,
                           int32_t n_steps, int32_t sampling_rate, float f_sigma_stop, double *epot_series,
                           double *ekin_series, double *sigma_e_series, double *sigma_f_max_series, float *f_var_last,
                           int32_t *n_steps_done, int32_t *n_samples, int32_t *n_rebuilds, void *cuda_stream) {
    if (!s || !positions || !velocities || !masses || n_steps < 0 || sampling_rate < 1 || !(dt_fs > 0.f) ||
        (n_steps >= sampling_rate && (!sigma_e_series || !sigma_f_max_series))) {
        set_error("gmnn_md_ensemble_steps: bad argument");
        return GMNN_INVALID_ARG;
    }
    if (int rcd = check_device(s->device, "gmnn_md_ensemble_steps")) return rcd;
    if (!s->have_list) {
        set_error("no neighbour list: call gmnn_build_neighbors first");
        return GMNN_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int64_t N = s->N;
    int rc;
    if (!s->ens_scratch && (rc = dev_alloc(&s->ens_scratch, (size_t)11 * N))) return rc;
    float *const f_keep = s->ens_scratch, *const e_mean = f_keep + 3 * N, *const e_var = e_mean + N,
                 *const f_mean = e_var + N, *const f_var = f_mean + 3 * N;
    double *const sig_e = s->e_total + 2;
    int32_t *const sig_f_bits = (int32_t *)(s->e_total + 3);
    const int keep_continue = s->md_continue;
    int32_t done = 0, samples = 0, rebuilds = 0;
    bool stopped = false;
    rc = GMNN_OK;
    while (done < n_steps && !stopped) {
        // the cheap mode (left-hand side of Eq. 6): sampling_rate steps on the mean energy, one backward each
        const int32_t chunk = (n_steps - done < sampling_rate) ? n_steps - done : sampling_rate;
        int32_t nreb = 0;
        s->md_continue = (done > 0) ? 1 : keep_continue;
        rc = gmnn_md_verlet_steps(s, positions, velocities, masses, dt_fs, chunk, epot_series ? epot_series + done : nullptr,
                                  ekin_series ? ekin_series + done : nullptr, &nreb, cuda_stream);
        if (rc) break;
        done += chunk;
        rebuilds += nreb;
        if (chunk < sampling_rate) break;
        // the expensive mode (right-hand side): one backward per head at the current positions.  The pass
        // borrows f_tmp; the mean-energy forces of the last step are put back afterwards so that the
        // trajectory is bit-for-bit the one without samples.
        GMNN_CUDA(cudaMemcpyAsync(f_keep, s->f_tmp, sizeof(float) * 3 * N, cudaMemcpyDeviceToDevice, st));
        if ((rc = ensemble_pass(s, positions, e_mean, e_var, f_mean, f_var, st))) break;
        if ((rc = launch_uncertainty_scalars(s, f_var, sig_e, sig_f_bits, st))) break;
        GMNN_CUDA(cudaMemcpyAsync(s->f_tmp, f_keep, sizeof(float) * 3 * N, cudaMemcpyDeviceToDevice, st));
        if (f_var_last) GMNN_CUDA(cudaMemcpyAsync(f_var_last, f_var, sizeof(float) * 3 * N, cudaMemcpyDeviceToDevice, st));
        double se = 0.0;
        float sf = 0.f;
        GMNN_CUDA(cudaMemcpyAsync(&se, sig_e, sizeof(double), cudaMemcpyDeviceToHost, st));
        GMNN_CUDA(cudaMemcpyAsync(&sf, sig_f_bits, sizeof(float), cudaMemcpyDeviceToHost, st));
        GMNN_CUDA(cudaStreamSynchronize(st));
        sigma_e_series[samples] = se;
        sigma_f_max_series[samples] = (double)sf;
        ++samples;
        if (f_sigma_stop > 0.f && sf > f_sigma_stop) stopped = true;
    }
    s->md_continue = keep_continue;
    if (n_steps_done) *n_steps_done = done;
    if (n_samples) *n_samples = samples;
    if (n_rebuilds) *n_rebuilds = rebuilds;
    return rc;
}

int gmnn_system_set_nose_hoover(gmnn_system *s, float temperature_K, float tau_fs, int32_t chain_length,
                                int32_t chain_steps, int32_t sy_steps) {
    if (!s) return GMNN_INVALID_ARG;
    s->md_state_valid = false;
    if (!(temperature_K > 0.f)) {  // off: NVE
        s->nhc_len = 0;
        return GMNN_OK;
    }
    if (!(tau_fs > 0.f) || !std::isfinite(tau_fs) || !std::isfinite(temperature_K) || chain_length < 1 ||
        chain_length > 8 || chain_steps < 1 || chain_steps > 16 || (sy_steps != 1 && sy_steps != 3 && sy_steps != 5)) {
        set_error("gmnn_system_set_nose_hoover: tau > 0, 1 <= chain_length <= 8, 1 <= chain_steps <= 16, sy_steps in {1, 3, 5}");
        return GMNN_INVALID_ARG;
    }
    if (s->lang_on) {
        set_error("a Langevin thermostat is set: switch it off first (one thermostat at a time)");
        return GMNN_INVALID_ARG;
    }
    int rc;
    if (!s->nhc && (rc = dev_alloc(&s->nhc, (size_t)26))) return rc;
    const double kT = 8.617333262e-5 * (double)temperature_K, tau = (double)tau_fs;
    double h[26] = {};
    for (int k = 0; k < chain_length; ++k) h[16 + k] = (k == 0 ? 3.0 * (double)s->N : 1.0) * kT * tau * tau;
    for (int k = chain_length; k < 8; ++k) h[16 + k] = 1.0;
    h[24] = 1.0;
    GMNN_CUDA(cudaMemcpy(s->nhc, h, sizeof(h), cudaMemcpyHostToDevice));
    if (!s->kT_now && (rc = dev_alloc(&s->kT_now, (size_t)1))) return rc;
    GMNN_CUDA(cudaMemcpy(s->kT_now, &kT, sizeof(double), cudaMemcpyHostToDevice));
    s->nhc_len = chain_length;
    s->nhc_chain_steps = chain_steps;
    s->nhc_sy_steps = sy_steps;
    s->nhc_kT = kT;
    return GMNN_OK;
}

int gmnn_system_get_nose_hoover(gmnn_system *s, double *xi, double *p_xi, double *thermostat_energy, void *cuda_stream) {
    if (!s || !xi || !p_xi || !thermostat_energy) return GMNN_INVALID_ARG;
    if (s->nhc_len == 0) {
        set_error("no Nose-Hoover chain is set");
        return GMNN_INVALID_ARG;
    }
    double h[26];
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GMNN_CUDA(cudaMemcpyAsync(h, s->nhc, sizeof(h), cudaMemcpyDeviceToHost, st));
    GMNN_CUDA(cudaStreamSynchronize(st));
    for (int k = 0; k < s->nhc_len; ++k) xi[k] = h[k], p_xi[k] = h[8 + k];
    *thermostat_energy = h[25];
    return GMNN_OK;
}

int gmnn_system_set_langevin(gmnn_system *s, float temperature_K, float gamma_per_fs, uint64_t seed, uint64_t first_step) {
    if (!s) return GMNN_INVALID_ARG;
    s->md_state_valid = false;
    if (!(temperature_K > 0.f)) {  // off
        s->lang_on = false;
        return GMNN_OK;
    }
    if (!(gamma_per_fs >= 0.f) || !std::isfinite(gamma_per_fs) || !std::isfinite(temperature_K)) {
        set_error("gmnn_system_set_langevin: gamma >= 0 (1/fs) and a finite temperature");
        return GMNN_INVALID_ARG;
    }
    if (s->nhc_len > 0) {
        set_error("a Nose-Hoover chain is set: switch it off first (one thermostat at a time)");
        return GMNN_INVALID_ARG;
    }
    int rc;
    if (!s->lang_step && (rc = dev_alloc(&s->lang_step, (size_t)1))) return rc;
    GMNN_CUDA(cudaMemcpy(s->lang_step, &first_step, sizeof(uint64_t), cudaMemcpyHostToDevice));
    s->lang_gamma = (double)gamma_per_fs;
    s->lang_kT = 8.617333262e-5 * (double)temperature_K;
    if (!s->kT_now && (rc = dev_alloc(&s->kT_now, (size_t)1))) return rc;
    GMNN_CUDA(cudaMemcpy(s->kT_now, &s->lang_kT, sizeof(double), cudaMemcpyHostToDevice));
    s->lang_seed = seed;
    s->lang_on = true;
    return GMNN_OK;
}

int gmnn_system_set_temperature_schedule(gmnn_system *s, int32_t n_points, const int64_t *steps, const float *temperatures_K) {
    if (!s || n_points < 0 || n_points > 64 || (n_points > 0 && (!steps || !temperatures_K))) {
        set_error("gmnn_system_set_temperature_schedule: 0 <= n_points <= 64 and non-null arrays");
        return GMNN_INVALID_ARG;
    }
    for (int k = 0; k < n_points; ++k)
        if (steps[k] < 0 || (k > 0 && steps[k] <= steps[k - 1]) || !(temperatures_K[k] > 0.f) || !std::isfinite(temperatures_K[k])) {
            set_error("temperature schedule: steps must ascend strictly from >= 0, temperatures must be positive");
            return GMNN_INVALID_ARG;
        }
    s->md_state_valid = false;
    s->sched_n = 0;
    if (n_points == 0) {  // back to the constant target of the thermostat that is set
        if (s->kT_now) {
            const double kT = s->lang_on ? s->lang_kT : s->nhc_kT;
            GMNN_CUDA(cudaMemcpy(s->kT_now, &kT, sizeof(double), cudaMemcpyHostToDevice));
        }
        return GMNN_OK;
    }
    int rc;
    if (!s->sched_steps) {
        if ((rc = dev_alloc(&s->sched_steps, (size_t)64))) return rc;
        if ((rc = dev_alloc(&s->sched_temps, (size_t)64))) return rc;
        if ((rc = dev_alloc(&s->sched_step, (size_t)1))) return rc;
    }
    if (!s->kT_now && (rc = dev_alloc(&s->kT_now, (size_t)1))) return rc;
    const uint64_t zero = 0;
    GMNN_CUDA(cudaMemcpy(s->sched_steps, steps, sizeof(int64_t) * n_points, cudaMemcpyHostToDevice));
    GMNN_CUDA(cudaMemcpy(s->sched_temps, temperatures_K, sizeof(float) * n_points, cudaMemcpyHostToDevice));
    GMNN_CUDA(cudaMemcpy(s->sched_step, &zero, sizeof(uint64_t), cudaMemcpyHostToDevice));
    s->sched_n = n_points;
    return GMNN_OK;
}

int gmnn_system_set_udd_bias(gmnn_system *s, float A, float B) {
    if (!s || !std::isfinite(A) || (A != 0.f && !(B > 0.f && std::isfinite(B)))) {
        set_error("gmnn_system_set_udd_bias: A must be finite and B > 0");
        return GMNN_INVALID_ARG;
    }
    ++g_config_gen;
    s->udd_A = A;
    if (A != 0.f) s->udd_B = B;
    s->md_state_valid = false;
    return GMNN_OK;
}

int gmnn_system_get_udd_bias(gmnn_system *s, double *e_bias, double *var_e, void *cuda_stream) {
    if (!s || !e_bias || !var_e) return GMNN_INVALID_ARG;
    double h[2] = {0.0, 0.0};
    if (s->udd_active) {
        cudaStream_t st = (cudaStream_t)cuda_stream;
        GMNN_CUDA(cudaMemcpyAsync(h, s->e_total + 4, sizeof(h), cudaMemcpyDeviceToHost, st));
        GMNN_CUDA(cudaStreamSynchronize(st));
    }
    *e_bias = h[0];
    *var_e = h[1];
    return GMNN_OK;
}

int gmnn_measure_fp32_peak(double *tflops, void *cuda_stream) {
    if (!tflops) return GMNN_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    GMNN_CUDA(cudaGetDevice(&dev));
    GMNN_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 8, iters = 4096;  // 8 blocks of 256 threads per SM: 16 warps per scheduler, 16 chains each
    float *scratch = nullptr;
    int rc = dev_alloc(&scratch, (size_t)blocks * 256);
    if (rc) return rc;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    rc = launch_fma_peak(blocks, 64, scratch, st);  // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 3 && !rc; ++rep) {
        cudaEventRecord(e0, st);
        rc = launch_fma_peak(blocks, iters, scratch, st);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) rc = GMNN_CUDA_ERROR;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tf = 2.0 * 128.0 * (double)iters * 256.0 * (double)blocks / ((double)ms * 1e-3) / 1e12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    dev_free(scratch);
    if (rc) return rc;
    *tflops = best;
    return GMNN_OK;
}

int gmnn_check(gmnn_system *s, void *cuda_stream) {
    if (!s) return GMNN_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = read_flags(s, st);
    if (rc) return rc;
    const int stale = s->flags_host[FLAG_STALE], oob = s->flags_host[FLAG_OUT_OF_BOX],
              over = s->flags_host[FLAG_MAXCOUNT] > s->cap;
    GMNN_CUDA(cudaMemsetAsync(s->flags, 0, sizeof(int32_t) * FLAG_WORDS, st));
    if (oob) {
        set_error("a position was outside [0, L) at a neighbour build");
        return GMNN_OUT_OF_BOX;
    }
    if (over) {
        set_error("neighbour list capacity exceeded");
        return GMNN_NEIGHBOR_OVERFLOW;
    }
    if (stale) {
        set_error("an atom moved more than skin/2 since the neighbour list was built");
        return GMNN_STALE_NEIGHBORS;
    }
    return GMNN_OK;
}

int gmnn_stage_times(gmnn_system *s, int32_t max_stages, const char **names, float *ms, int32_t *counts) {
    if (!s || !names || !ms) return GMNN_INVALID_ARG;
    const int n = s->n_stage_events;
    if (n < 2) return 0;
    GMNN_CUDA(cudaEventSynchronize(s->events[n - 1]));
    std::vector<const char *> uniq;
    std::vector<double> total;
    std::vector<int> cnt;
    for (int k = 1; k < n; ++k) {
        const char *nm = s->stage_names[k];
        if (!nm) continue;  // a begin() marker: the gap before it is not a stage
        float t = 0.f;
        GMNN_CUDA(cudaEventElapsedTime(&t, s->events[k - 1], s->events[k]));
        size_t u = 0;
        for (; u < uniq.size(); ++u)
            if (!strcmp(uniq[u], nm)) break;
        if (u == uniq.size()) {
            uniq.push_back(nm);
            total.push_back(0.0);
            cnt.push_back(0);
        }
        total[u] += t;
        cnt[u] += 1;
    }
    int k = 0;
    for (; k < (int)uniq.size() && k < max_stages; ++k) {
        names[k] = uniq[k];
        ms[k] = (float)(total[k] / cnt[k]);
        if (counts) counts[k] = cnt[k];
    }
    return k;
}

int gmnn_debug_read(gmnn_system *s, const char *name, void *dst, int64_t bytes) {
    if (!s || !name || !dst) return GMNN_INVALID_ARG;
    const int64_t N = s->N;
    const gmnn_model *m = s->model;
    const void *src = nullptr;
    int64_t need = 0;
    if (!strcmp(name, "perm")) { src = s->perm; need = 4 * N; }
    else if (!strcmp(name, "count")) { src = s->count; need = 4 * N; }
    else if (!strcmp(name, "xref")) { src = s->xref; need = 4 * 3 * N; }
    else if (!strcmp(name, "psi")) { src = s->psi; need = 4 * N * m->hp.n_radial * PSI; }
    else if (!strcmp(name, "A")) { src = s->A; need = 4 * N * m->hp.n_radial * PSI; }
    else if (!strcmp(name, "G")) { src = s->G; need = 4 * N * m->n_features; }
    else if (!strcmp(name, "dG")) { src = s->dG; need = 4 * N * m->n_features; }
    else if (!strcmp(name, "e_heads")) { src = s->e_heads; need = 4 * N * m->hp.n_heads; }
    else if (!strcmp(name, "H0")) { src = s->H[0]; need = 4 * N * m->dims[1]; }
    else if (!strcmp(name, "D0")) { src = s->D[0]; need = 4 * N * m->dims[1]; }
    else {
        set_error("gmnn_debug_read: unknown array '%s'", name);
        return GMNN_INVALID_ARG;
    }
    if (bytes != need) {
        set_error("gmnn_debug_read('%s'): expected %lld bytes, got %lld", name, (long long)need, (long long)bytes);
        return GMNN_INVALID_ARG;
    }
    GMNN_CUDA(cudaDeviceSynchronize());
    // row-order arrays are handed back in internal atom order: row of atom k = mrow[k] (identity with one weight set)
    std::vector<int32_t> mrow;
    if (s->mrow) {
        mrow.resize((size_t)N);
        GMNN_CUDA(cudaMemcpy(mrow.data(), s->mrow, sizeof(int32_t) * (size_t)N, cudaMemcpyDeviceToHost));
    }
    auto row_of = [&](int64_t k) { return mrow.empty() ? k : (int64_t)mrow[(size_t)k]; };
    if (!strcmp(name, "dG") || !strcmp(name, "G") || !strcmp(name, "H0") || !strcmp(name, "D0")) {
        // stored as [rows/128][F][128] tiles: hand back [N][F]
        const int64_t F = need / (4 * N), tiles = (s->n_rows + 127) / 128;
        std::vector<float> tmp((size_t)(tiles * 128 * F));
        GMNN_CUDA(cudaMemcpy(tmp.data(), src, tmp.size() * 4, cudaMemcpyDeviceToHost));
        float *out = static_cast<float *>(dst);
        for (int64_t k = 0; k < N; ++k) {
            const int64_t i = row_of(k);
            for (int64_t f = 0; f < F; ++f) out[k * F + f] = tmp[(size_t)(((i >> 7) * F + f) * 128 + (i & 127))];
        }
        return GMNN_OK;
    }
    if (!mrow.empty() && (!strcmp(name, "psi") || !strcmp(name, "A"))) {
        const int64_t W = need / (4 * N);
        std::vector<float> tmp((size_t)(s->n_rows * W));
        GMNN_CUDA(cudaMemcpy(tmp.data(), src, tmp.size() * 4, cudaMemcpyDeviceToHost));
        float *out = static_cast<float *>(dst);
        for (int64_t k = 0; k < N; ++k) memcpy(out + k * W, tmp.data() + (size_t)(row_of(k) * W), (size_t)W * 4);
        return GMNN_OK;
    }
    GMNN_CUDA(cudaMemcpy(dst, src, (size_t)bytes, cudaMemcpyDeviceToHost));
    return GMNN_OK;
}

}  // extern "C"
