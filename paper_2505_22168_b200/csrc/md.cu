// md.cu -- output scatter, fixed-order fp64 reductions, velocity-Verlet kicks and drift with the
// skin test, and the ensemble statistics (Eq. 5,
// :169-171 MD loop on the device, :367 dt, :381 skin).
#include "gmnn_internal.h"

namespace gmnn {

constexpr double ACC_CONV = 9.648533212e-3;  // (eV/Ang/amu) -> Ang/fs^2
constexpr int RED_BLOCKS = 1024;             // partial sums of the two-stage reductions

static inline unsigned nblocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }

// internal (cell-sorted) order -> caller order
__global__ void k_scatter(int64_t N, const int32_t *__restrict__ perm, const float *__restrict__ e_int,
                          const float *__restrict__ f_int, float *e_out, float *f_out) {
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int64_t i = perm[k];
    if (e_out) e_out[i] = e_int[k];
    if (f_out) {
        f_out[3 * i] = f_int[3 * k];
        f_out[3 * i + 1] = f_int[3 * k + 1];
        f_out[3 * i + 2] = f_int[3 * k + 2];
    }
}

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    v = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : 0.0;
    if (wid == 0) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    }
    __syncthreads();
    return v;  // valid in thread 0
}

// stage 1: block b sums a fixed contiguous slice in a fixed order; stage 2: one block sums the
// partials.  The result depends on N only, never on scheduling.
__global__ void __launch_bounds__(256) k_sum_stage1(int64_t N, const float *__restrict__ x, double *partial) {
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t b = blockIdx.x * per, e = (b + per < N) ? b + per : N;
    double v = 0.0;
    for (int64_t q = b + threadIdx.x; q < e; q += blockDim.x) v += (double)x[q];
    v = block_sum(v);
    if (threadIdx.x == 0) partial[blockIdx.x] = v;
}

__global__ void __launch_bounds__(256) k_ke_stage1(int64_t N, const float *__restrict__ v, const float *__restrict__ m,
                                                  double *partial) {
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t b = blockIdx.x * per, e = (b + per < N) ? b + per : N;
    double acc = 0.0;
    for (int64_t q = b + threadIdx.x; q < e; q += blockDim.x) {
        const double vx = v[3 * q], vy = v[3 * q + 1], vz = v[3 * q + 2];
        acc += 0.5 * (double)m[q] * (vx * vx + vy * vy + vz * vz);
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}

__global__ void __launch_bounds__(256) k_sum_stage2(int n, const double *__restrict__ partial, double factor, double *out, double *out2,
                                                    const double *__restrict__ add) {
    double v = 0.0;
    for (int q = threadIdx.x; q < n; q += blockDim.x) v += partial[q];
    v = block_sum(v);
    if (threadIdx.x == 0) {
        v = v * factor + (add ? *add : 0.0);  // add: the UDD bias of this evaluation (Eq. 9)
        *out = v;
        if (out2) *out2 = v;
    }
}

// v += (dt/2) a;  x += dt v;  squared displacement from the build positions -> max into flags.
__global__ void __launch_bounds__(256)
k_kick_drift(int64_t N, float *x, float *v, const float *__restrict__ f, const float *__restrict__ m, float dt,
             const float *__restrict__ xref, int32_t *flags) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    float d2 = 0.f;
    if (i < N) {
        const float c = 0.5f * dt * (float)ACC_CONV / m[i];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float vv = fmaf(c, f[3 * i + a], v[3 * i + a]);
            float xx = fmaf(dt, vv, x[3 * i + a]);
            v[3 * i + a] = vv;
            x[3 * i + a] = xx;
            const float d = xx - xref[3 * i + a];
            d2 = fmaf(d, d, d2);
        }
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, o));
    if ((threadIdx.x & 31) == 0 && d2 > 0.f) atomicMax(&flags[FLAG_DISP2], __float_as_int(d2));  // d2 >= 0: int order = float order
}

__global__ void __launch_bounds__(256)
k_kick(int64_t N, float *v, const float *__restrict__ f, const float *__restrict__ m, float dt) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float c = 0.5f * dt * (float)ACC_CONV / m[i];
#pragma unroll
    for (int a = 0; a < 3; ++a) v[3 * i + a] = fmaf(c, f[3 * i + a], v[3 * i + a]);
}

// Welford update in head order: after head h (0-based), mean/M2 of heads 0..h.
__global__ void k_finish_var(int64_t n, float *m2, float inv_heads) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < n) m2[t] *= inv_heads;
}

// per-atom energy mean / population variance over the heads (Eq. 5 with 1/N_ens), caller order
__global__ void k_energy_stats(int64_t N, int M, const int32_t *__restrict__ perm, const float *__restrict__ e_heads,
                               float *e_mean, float *e_var) {
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= N) return;
    const float *e = e_heads + k * (int64_t)M;
    float mu = 0.f;
    for (int m = 0; m < M; ++m) mu += e[m];
    mu /= (float)M;
    float var = 0.f;
    for (int m = 0; m < M; ++m) var = fmaf(e[m] - mu, e[m] - mu, var);
    const int64_t i = perm[k];
    e_mean[i] = mu;
    e_var[i] = var / (float)M;
}

int launch_scatter_outputs(gmnn_system *s, float *e_atom_out, float *forces_out, cudaStream_t st) {
    k_scatter<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, s->perm, s->e_atom, s->f_int, e_atom_out, forces_out);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

static int red_blocks(int64_t N) { return (int)(N < RED_BLOCKS * 256 ? (N + 255) / 256 : RED_BLOCKS); }

int launch_energy_sum(gmnn_system *s, double *energy_out, cudaStream_t st, double *energy_out2) {
    const int nb = red_blocks(s->N);
    k_sum_stage1<<<nb, 256, 0, st>>>(s->N, s->e_atom, s->partial);
    GMNN_LAUNCHED();
    k_sum_stage2<<<1, 256, 0, st>>>(nb, s->partial, 1.0, energy_out, energy_out2, s->udd_active ? s->e_total + 4 : nullptr);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// virial: component c = blockIdx.y of vir_atom [9][N]; same fixed two-stage order as the energy sum
__global__ void __launch_bounds__(256) k_sum9_stage1(int64_t N, const float *__restrict__ x, double *partial) {
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t b = blockIdx.x * per, e = b + per < N ? b + per : N;
    const float *xc = x + (int64_t)blockIdx.y * N;
    double v = 0.0;
    for (int64_t q = b + threadIdx.x; q < e; q += blockDim.x) v += (double)xc[q];
    v = block_sum(v);
    if (threadIdx.x == 0) partial[blockIdx.y * gridDim.x + blockIdx.x] = v;
}
__global__ void __launch_bounds__(256) k_sum9_stage2(int n, const double *__restrict__ partial, double *out) {
    double v = 0.0;
    for (int q = threadIdx.x; q < n; q += blockDim.x) v += partial[blockIdx.x * n + q];
    v = block_sum(v);
    if (threadIdx.x == 0) out[blockIdx.x] = v;
}

int launch_virial_sum(gmnn_system *s, double *virial_out, cudaStream_t st) {
    const int nb = red_blocks(s->N) < 113 ? red_blocks(s->N) : 113;  // 9 x 113 partials fit the 2048-double scratch
    k_sum9_stage1<<<dim3(nb, 9), 256, 0, st>>>(s->N, s->vir_atom, s->partial);
    GMNN_LAUNCHED();
    k_sum9_stage2<<<9, 256, 0, st>>>(nb, s->partial, virial_out);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_ke(gmnn_system *s, const float *v, const float *m, double *ekin_out, cudaStream_t st, double *ekin_out2) {
    const int nb = red_blocks(s->N);
    k_ke_stage1<<<nb, 256, 0, st>>>(s->N, v, m, s->partial + RED_BLOCKS);
    GMNN_LAUNCHED();
    k_sum_stage2<<<1, 256, 0, st>>>(nb, s->partial + RED_BLOCKS, 1.0 / ACC_CONV, ekin_out, ekin_out2, nullptr);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_kick_drift(gmnn_system *s, float *x, float *v, const float *f, const float *m, float dt, cudaStream_t st) {
    k_kick_drift<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, x, v, f, m, dt, s->xref, s->flags);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_kick_ke(gmnn_system *s, float *v, const float *f, const float *m, float dt, double *ekin_out, cudaStream_t st,
                   double *ekin_out2) {
    k_kick<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, v, f, m, dt);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    if (ekin_out) return launch_ke(s, v, m, ekin_out, st, ekin_out2);
    return GMNN_OK;
}

// Series output of the MD loop with a device-side step counter, so that every step issues the same
// launches with the same arguments (the loop body is replayed as a CUDA graph).
__global__ void k_series_append(const double *__restrict__ e_total, double *epot_series, double *ekin_series,
                                int32_t *counter) {
    const int32_t k = *counter;
    if (epot_series) epot_series[k] = e_total[0];
    if (ekin_series) ekin_series[k] = e_total[1];
    *counter = k + 1;
}
__global__ void k_set_int(int32_t *p, int32_t v) { *p = v; }

int launch_series_append(gmnn_system *s, double *epot_series, double *ekin_series, cudaStream_t st) {
    k_series_append<<<1, 1, 0, st>>>(s->e_total, epot_series, ekin_series, s->flags + FLAG_MD_STEP);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_series_reset(gmnn_system *s, int32_t next_index, cudaStream_t st) {
    k_set_int<<<1, 1, 0, st>>>(s->flags + FLAG_MD_STEP, next_index);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_finish_var(int64_t n, float *m2, int n_heads, cudaStream_t st) {
    k_finish_var<<<nblocks(n, 256), 256, 0, st>>>(n, m2, 1.f / (float)n_heads);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_ensemble_energy_stats(gmnn_system *s, float *e_mean, float *e_var, cudaStream_t st) {
    k_energy_stats<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, s->model->dims[s->model->hp.n_hidden + 1], s->perm,
                                                       s->e_heads, e_mean, e_var);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// ---- uncertainty scalars of a switching-mode sample (SURVEY 8(f) NEXT-1; PAPER.md:75-77 Eq. 5, :71, :175) ----
// Total energy of every head, E^(m) = sum_i E_i^(m), in fp64 and in a fixed order: block (b, m) sums
// head m over a contiguous slice of atoms, one block per head adds the slices.
__global__ void __launch_bounds__(256) k_head_totals_stage1(int64_t N, int M, const float *__restrict__ e_heads,
                                                            double *partial) {
    const int m = blockIdx.y;
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t b = blockIdx.x * per, e = (b + per < N) ? b + per : N;
    double v = 0.0;
    for (int64_t q = b + threadIdx.x; q < e; q += blockDim.x) v += (double)e_heads[q * M + m];
    v = block_sum(v);
    if (threadIdx.x == 0) partial[(int64_t)m * gridDim.x + blockIdx.x] = v;
}

// sigma_E = sqrt(1/M sum_m (E^(m) - mean)^2): one block, thread m owns head m (M <= 64)
__global__ void __launch_bounds__(64) k_sigma_e(int nb, int M, const double *__restrict__ partial, double *out) {
    __shared__ double tot[64];
    const int m = threadIdx.x;
    if (m < M) {
        double v = 0.0;
        for (int b = 0; b < nb; ++b) v += partial[(int64_t)m * nb + b];
        tot[m] = v;
    }
    __syncthreads();
    if (m == 0) {
        double mean = 0.0, var = 0.0;
        for (int q = 0; q < M; ++q) mean += tot[q];
        mean /= (double)M;
        for (int q = 0; q < M; ++q) var += (tot[q] - mean) * (tot[q] - mean);
        *out = sqrt(var / (double)M);
    }
}

// max_i sqrt(f_var[i][x] + f_var[i][y] + f_var[i][z]); a maximum of non-negative floats does not depend
// on the order, so an integer atomicMax on the bit pattern keeps the result deterministic
__global__ void __launch_bounds__(256) k_sigma_f_max(int64_t N, const float *__restrict__ f_var, int32_t *out_bits) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    float v = 0.f;
    if (i < N) v = sqrtf(f_var[3 * i] + f_var[3 * i + 1] + f_var[3 * i + 2]);
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0 && v > 0.f) atomicMax(out_bits, __float_as_int(v));
}

// UDD bias (Eq. 9) on the head totals of stage 1:
//   E_b = A [exp(-s2 / (M N B^2)) - 1],  s2 = 1/M sum_m (E^(m) - mean)^2  (Eq. 5 on total energies, reading R27)
// The gradient of mean + E_b is sum_m c_m grad E^(m) with  c_m = 1/M + E_b'(s2) 2/M (E^(m) - mean)  (the
// weights of the -mean term sum to zero), so ONE backward pass with head weights c gives the biased forces.
__global__ void __launch_bounds__(64) k_udd_weights(int nb, int M, const double *__restrict__ partial, double A, double B,
                                                    double n_atoms, float *head_w, double *scal) {
    __shared__ double tot[64];
    const int m = threadIdx.x;
    if (m < M) {
        double v = 0.0;
        for (int b = 0; b < nb; ++b) v += partial[(int64_t)m * nb + b];
        tot[m] = v;
    }
    __syncthreads();
    double mean = 0.0, var = 0.0;
    for (int q = 0; q < M; ++q) mean += tot[q];
    mean /= (double)M;
    for (int q = 0; q < M; ++q) var += (tot[q] - mean) * (tot[q] - mean);
    var /= (double)M;
    const double width = (double)M * n_atoms * B * B;
    const double ex = exp(-var / width);
    if (m < M) head_w[m] = (float)(1.0 / M + (-A / width * ex) * (2.0 / M) * (tot[m] - mean));
    if (m == 0) {
        scal[0] = A * (ex - 1.0);
        scal[1] = var;
    }
}

static int head_total_blocks(const gmnn_system *s) {
    const int M = s->model->hp.n_heads;
    int nb = red_blocks(s->N);
    if (nb * M > 2 * RED_BLOCKS) nb = 2 * RED_BLOCKS / M;  // partial holds 2 * RED_BLOCKS doubles
    return nb;
}

// head_w_out [M] <- c;  scal[0] <- E_b, scal[1] <- sigma_E^2  (from e_heads of the forward just run)
int launch_udd_weights(gmnn_system *s, float *head_w_out, double *scal, cudaStream_t st) {
    const int M = s->model->hp.n_heads, nb = head_total_blocks(s);
    k_head_totals_stage1<<<dim3(nb, M), 256, 0, st>>>(s->N, M, s->e_heads, s->partial);
    GMNN_LAUNCHED();
    k_udd_weights<<<1, 64, 0, st>>>(nb, M, s->partial, (double)s->udd_A, (double)s->udd_B, (double)s->N, head_w_out, scal);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// out: double sigma_e at out_d[0]; float bits of sigma_f_max at out_bits[0] (zeroed here first)
int launch_uncertainty_scalars(gmnn_system *s, const float *f_var, double *out_d, int32_t *out_bits, cudaStream_t st) {
    const int M = s->model->hp.n_heads, nb = head_total_blocks(s);
    GMNN_CUDA(cudaMemsetAsync(out_bits, 0, sizeof(int32_t), st));
    k_head_totals_stage1<<<dim3(nb, M), 256, 0, st>>>(s->N, M, s->e_heads, s->partial);
    GMNN_LAUNCHED();
    k_sigma_e<<<1, 64, 0, st>>>(nb, M, s->partial, out_d);
    GMNN_LAUNCHED();
    k_sigma_f_max<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, f_var, out_bits);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// ---- NVT: Nose-Hoover chain (PAPER.md:365-375 thermostat_chain) ----
// The chain operator of Martyna, Tuckerman, Tobias and Klein for half a time step, on the device so that the
// thermostatted step stays one replayable launch sequence: one thread, fp64, reads the kinetic energy the
// last kick left in ek, updates (xi, p_xi), and leaves the velocity scale factor for k_scale_v.
// st: [0, 8) xi, [8, 16) p_xi, [16, 24) Q, [24] scale factor, [25] thermostat energy
__global__ void k_nhc_half(double *ek, double *st, int Mc, int chain_steps, int sy_steps, double dof,
                           const double *__restrict__ kT_now, double dt) {
    const double kT = *kT_now;  // the step's target (constant, or this step's value of the temperature schedule)
    double *xi = st, *pxi = st + 8;
    const double *Q = st + 16;
    double w[5];
    if (sy_steps == 3) {
        const double a = 1.0 / (2.0 - cbrt(2.0));
        w[0] = a, w[1] = 1.0 - 2.0 * a, w[2] = a;
    } else if (sy_steps == 5) {
        const double a = 1.0 / (4.0 - cbrt(4.0));
        w[0] = w[1] = w[3] = w[4] = a, w[2] = 1.0 - 4.0 * a;
    } else {
        w[0] = 1.0;
    }
    double ke2 = 2.0 * *ek, scale = 1.0;
    const double delta = dt / chain_steps;
    for (int c = 0; c < chain_steps; ++c)
        for (int y = 0; y < sy_steps; ++y) {
            const double d2 = delta * w[y] / 2, d4 = delta * w[y] / 4, d8 = delta * w[y] / 8;
            double G = (Mc > 1) ? pxi[Mc - 2] * pxi[Mc - 2] / Q[Mc - 2] - kT : ke2 - dof * kT;
            pxi[Mc - 1] += d4 * G;
            for (int k = Mc - 2; k >= 0; --k) {
                G = (k == 0) ? ke2 - dof * kT : pxi[k - 1] * pxi[k - 1] / Q[k - 1] - kT;
                const double e = exp(-d8 * pxi[k + 1] / Q[k + 1]);
                pxi[k] = e * (e * pxi[k] + d4 * G);
            }
            const double e0 = exp(-d2 * pxi[0] / Q[0]);
            scale *= e0;
            ke2 *= e0 * e0;
            for (int k = 0; k < Mc; ++k) xi[k] += d2 * pxi[k] / Q[k];
            G = ke2 - dof * kT;
            for (int k = 0; k < Mc - 1; ++k) {
                const double e = exp(-d8 * pxi[k + 1] / Q[k + 1]);
                pxi[k] = e * (e * pxi[k] + d4 * G);
                G = pxi[k] * pxi[k] / Q[k] - kT;
            }
            pxi[Mc - 1] += d4 * G;
        }
    *ek = 0.5 * ke2;
    st[24] = scale;
    double et = dof * kT * xi[0];
    for (int k = 0; k < Mc; ++k) et += pxi[k] * pxi[k] / (2.0 * Q[k]) + (k > 0 ? kT * xi[k] : 0.0);
    st[25] = et;
}

__global__ void __launch_bounds__(256) k_scale_v(int64_t n3, float *v, const double *__restrict__ scale) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < n3) v[t] *= (float)*scale;
}

// chain operator for dt/2 on the kinetic energy in ek (updated), then v *= scale
int launch_nhc_half(gmnn_system *s, float *v, double *ek, float dt, cudaStream_t st) {
    k_nhc_half<<<1, 1, 0, st>>>(ek, s->nhc, s->nhc_len, s->nhc_chain_steps, s->nhc_sy_steps, 3.0 * (double)s->N, s->kT_now,
                                (double)dt);
    GMNN_LAUNCHED();
    k_scale_v<<<nblocks(3 * s->N, 256), 256, 0, st>>>(3 * s->N, v, s->nhc + 24);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// ---- Langevin dynamics, BAOAB (reading R29) ----
__device__ __forceinline__ uint64_t splitmix64_at(uint64_t seed, uint64_t counter) {
    uint64_t z = seed + (counter + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// B A O A of one step (the closing B is k_kick): replaces k_kick_drift, skin test included.  The three normals of
// atom i at step t come from splitmix64 outputs (t N + i) 2 + {0, 1}, Box-Muller in fp64 (the same definition the
// oracle implements on its own), so the trajectory does not depend on the launch geometry or on replay.
__global__ void __launch_bounds__(256)
k_baoab(int64_t N, float *x, float *v, const float *__restrict__ f, const float *__restrict__ m, float dt, double c1,
        const double *__restrict__ kT_now, uint64_t seed, const uint64_t *__restrict__ step, const float *__restrict__ xref,
        int32_t *flags) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    float d2 = 0.f;
    if (i < N) {
        const double kT_acc = *kT_now * ACC_CONV;  // the step's target temperature (see k_nhc_half)
        const uint64_t base = (*step * (uint64_t)N + (uint64_t)i) * 2ull;
        const uint64_t w0 = splitmix64_at(seed, base), w1 = splitmix64_at(seed, base + 1ull);
        const double two32 = 1.0 / 4294967296.0, twopi = 6.283185307179586476925286766559;
        const double u1 = ((double)(uint32_t)w0 + 1.0) * two32, u2 = ((double)(uint32_t)(w0 >> 32) + 1.0) * two32;
        const double u3 = ((double)(uint32_t)w1 + 1.0) * two32, u4 = ((double)(uint32_t)(w1 >> 32) + 1.0) * two32;
        const double r1 = sqrt(-2.0 * log(u1)), r2 = sqrt(-2.0 * log(u3));
        double sn, cs;
        sincos(twopi * u2, &sn, &cs);
        const double xi[3] = {r1 * cs, r1 * sn, r2 * cos(twopi * u4)};
        const float mi = m[i];
        const float c = 0.5f * dt * (float)ACC_CONV / mi;
        const float c2 = (float)sqrt(kT_acc * (1.0 - c1 * c1) / (double)mi);
        const float hdt = 0.5f * dt, c1f = (float)c1;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float vv = fmaf(c, f[3 * i + a], v[3 * i + a]);
            float xx = fmaf(hdt, vv, x[3 * i + a]);
            vv = fmaf(c1f, vv, c2 * (float)xi[a]);
            xx = fmaf(hdt, vv, xx);
            v[3 * i + a] = vv;
            x[3 * i + a] = xx;
            const float d = xx - xref[3 * i + a];
            d2 = fmaf(d, d, d2);
        }
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, o));
    if ((threadIdx.x & 31) == 0 && d2 > 0.f) atomicMax(&flags[FLAG_DISP2], __float_as_int(d2));
}

__global__ void k_inc_u64(uint64_t *p) { *p += 1ull; }

// Temperature schedule (reading R32): k_B T of MD step *step, piecewise linear between
// the points, constant before the first and after the last; then the step counter moves on.  One thread.
__global__ void k_schedule_eval(int n, const int64_t *__restrict__ steps, const float *__restrict__ temps, uint64_t *step,
                                double *kT_now) {
    const double t = (double)*step;
    double T = (double)temps[n - 1];
    if (t <= (double)steps[0]) {
        T = (double)temps[0];
    } else {
        for (int k = 1; k < n; ++k)
            if (t <= (double)steps[k]) {
                const double a = (t - (double)steps[k - 1]) / ((double)steps[k] - (double)steps[k - 1]);
                T = (double)temps[k - 1] + a * ((double)temps[k] - (double)temps[k - 1]);
                break;
            }
    }
    *kT_now = 8.617333262e-5 * T;
    *step += 1ull;
}

int launch_schedule_eval(gmnn_system *s, cudaStream_t st) {
    k_schedule_eval<<<1, 1, 0, st>>>(s->sched_n, s->sched_steps, s->sched_temps, s->sched_step, s->kT_now);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_baoab(gmnn_system *s, float *x, float *v, const float *f, const float *m, float dt, cudaStream_t st) {
    const double c1 = exp(-s->lang_gamma * (double)dt);
    k_baoab<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, x, v, f, m, dt, c1, s->kT_now, s->lang_seed, s->lang_step, s->xref,
                                                 s->flags);
    GMNN_LAUNCHED();
    k_inc_u64<<<1, 1, 0, st>>>(s->lang_step);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}


// ---- calibration: the fp32 FMA rate this GPU sustains right now (bench.py's "alu" roof, measured in the same run) ----
// Every thread runs 16 independent dependent-FMA chains (registers only); 2 flop per FMA.  The result is stored so that
// nothing is optimised away.
__global__ void __launch_bounds__(256) k_fma_peak(int iters, float seed, float *out) {
    float a[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) a[q] = seed + (float)(threadIdx.x + q);
    const float b = 1.0000001f, c = 1e-7f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int q = 0; q < 16; ++q) a[q] = fmaf(a[q], b, c);
    }
    float sum = 0.f;
#pragma unroll
    for (int q = 0; q < 16; ++q) sum += a[q];
    if (sum == 12345.678f) out[blockIdx.x * blockDim.x + threadIdx.x] = sum;  // practically never: keeps the chains alive
}

int launch_fma_peak(int blocks, int iters, float *scratch, cudaStream_t st) {
    k_fma_peak<<<blocks, 256, 0, st>>>(iters, 1.0f, scratch);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

}  // namespace gmnn

// ---------------------------------------------------------------------------------------------------------------------
// gmnn_sum_energies_static (include/gmnn.h): the two-stage fp64 sum of per-atom energies (stage 1 / stage 2 above,
// the kernels behind the total energy of every evaluation) for callers that may not allocate: the block partials
// that launch_energy_sum keeps in a cudaMalloc'ed buffer of the system live here in a file-scope device array.
// Every GPU that loads the library holds these 8 KB until exit.  Every call shares them: stage 1 overwrites the
// slots [0, blocks) that stage 2 of the same call reads, so nothing has to start at zero and stale contents of an
// earlier call are never read; calls that overlap on the GPU (two streams, two host threads) race on them.
// ---------------------------------------------------------------------------------------------------------------------
namespace gmnn {
constexpr int64_t STATIC_SUM_MAX_ATOMS = (int64_t)RED_BLOCKS * 256 * 64;  // 16 777 216 = GMNN_STATIC_SUM_MAX_ATOMS
static_assert(STATIC_SUM_MAX_ATOMS == GMNN_STATIC_SUM_MAX_ATOMS, "include/gmnn.h states the limit");
static __device__ __align__(256) double g_static_partial[RED_BLOCKS];
// In host code the name g_static_partial is a host-side stand-in, not a device address: the address the kernels get
// is looked up once per device, with that device current.
static double *g_static_partial_dev[MAX_DEVICES] = {};

static int static_partial_ptr(double **ptr) {
    const int dev = current_device();
    if (!g_static_partial_dev[dev]) {
        void *p = nullptr;
        GMNN_CUDA(cudaGetSymbolAddress(&p, g_static_partial));
        g_static_partial_dev[dev] = static_cast<double *>(p);
    }
    *ptr = g_static_partial_dev[dev];
    return GMNN_OK;
}
}  // namespace gmnn

extern "C" int gmnn_sum_energies_static(const float *e_atom, int64_t n_atoms, double *energy, void *cuda_stream) {
    using namespace gmnn;
    if (!e_atom || !energy || n_atoms < 0) {
        set_error("gmnn_sum_energies_static: null pointer or negative atom count");
        return GMNN_INVALID_ARG;
    }
    if (n_atoms > STATIC_SUM_MAX_ATOMS) {
        set_error("gmnn_sum_energies_static: %lld atoms exceed the static scratch limit of %lld "
                  "(GMNN_STATIC_SUM_MAX_ATOMS); use gmnn_energy_forces' own total instead",
                  (long long)n_atoms, (long long)STATIC_SUM_MAX_ATOMS);
        return GMNN_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *partial = nullptr;
    int rc = static_partial_ptr(&partial);
    if (rc) return rc;
    const int nb = red_blocks(n_atoms);
    if (nb > 0) {
        k_sum_stage1<<<nb, 256, 0, st>>>(n_atoms, e_atom, partial);
        GMNN_LAUNCHED();
    }
    k_sum_stage2<<<1, 256, 0, st>>>(nb, partial, 1.0, energy, nullptr, nullptr);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}
