// mlp_simt.cu -- the per-atom MLP readout and its input gradient in plain fp32 FMA
// (SURVEY.md 8(a) rows a7, a8; PAPER.md:63-65 Eq. 4, :151 ensemble axis, :153 forces by gradient).
// This is mlp_precision = GMNN_MLP_FP32: the reference-precision path (fp32 tolerance of
// north_star).  The tcgen05 tensor-core variants live in mlp_tc.cu.
//
// Forward, layer l (weights W[l] : [dims[l]][dims[l+1]]):
//     z = X W[l] + b[l];  H[l] = swish(z);  D[l] = swish'(z)          (both stored: D feeds the backward)
// Heads:  y_m = H_last . W_last[:, m] + b_last[m];  E_i^(m) = sigma_Z y_m + mu_Z
// Backward of E_c = sum_m c_m E^(m), WITHOUT the per-atom factor sigma_Z (applied later, the
// chain is linear in it):  v = W_last c;  dZ_last = D_last * v  is folded into the weights,
//     dH = D_last (diag(v) W^T),  dZ = dH * D[l-1], ...,  dG = dZ_1 W[0]^T.
//
// GEMM kernel: 128x128x8 tiles, 256 threads, 8x8 outputs per thread, double-buffered shared
// memory with register prefetch, A tile stored transposed so both operands are read as float4.
#include "gmnn_internal.h"

namespace gmnn {

enum { EPI_PLAIN = 0, EPI_HIDDEN = 1, EPI_MUL = 2 };

__device__ __forceinline__ void swish_pair(float z, float &h, float &d) {
    const float s = 1.f / (1.f + __expf(-z));
    h = z * s;
    d = s * (1.f + z * (1.f - s));
}

constexpr int BM = 128, BN = 128, BK = 8, APITCH = 132;

// C = A . B with A, C, C2, Dmul tile-transposed ([M/128][cols][128], padded to whole tiles, the layout
// every MLP matrix uses: see mlp_tc.cu) and B = W[l] row-major [K][N].
template <int EPI>
__global__ void __launch_bounds__(256)
k_sgemm(int M, int N, int K, const float *__restrict__ At, const float *__restrict__ B, int ldb,
        float *__restrict__ Ct, const float *__restrict__ bias, float *__restrict__ C2t,
        const float *__restrict__ Dmult) {
    __shared__ __align__(16) float As[2][BK][APITCH];
    __shared__ __align__(16) float Bs[2][BK][BN];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int n0 = blockIdx.x * BN;
    const int ak = tid >> 5, ar = (tid & 31) * 4;  // A tile: k row, first of this thread's 4 atoms
    const int bk = tid >> 5, bc = (tid & 31) * 4;  // B tile: k row, column of this thread's float4
    const bool b_ok = (n0 + bc) < N;
    const float *Ap = At + ((int64_t)blockIdx.y * K + ak) * BM + ar;
    const float *Bp = B + (int64_t)bk * ldb + n0 + bc;
    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;

    const int nk = K / BK;
    float4 ra = __ldg(reinterpret_cast<const float4 *>(Ap));
    float4 rb = b_ok ? __ldg(reinterpret_cast<const float4 *>(Bp)) : make_float4(0.f, 0.f, 0.f, 0.f);
    *reinterpret_cast<float4 *>(&As[0][ak][ar]) = ra;
    *reinterpret_cast<float4 *>(&Bs[0][bk][bc]) = rb;
    __syncthreads();
    int cur = 0;
    for (int kt = 0; kt < nk; ++kt) {
        if (kt + 1 < nk) {
            ra = __ldg(reinterpret_cast<const float4 *>(Ap + (int64_t)(kt + 1) * BK * BM));
            rb = b_ok ? __ldg(reinterpret_cast<const float4 *>(Bp + (int64_t)(kt + 1) * BK * ldb)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int kk = 0; kk < BK; ++kk) {
            const float4 a0 = *reinterpret_cast<const float4 *>(&As[cur][kk][ty * 4]);
            const float4 a1 = *reinterpret_cast<const float4 *>(&As[cur][kk][64 + ty * 4]);
            const float4 b0 = *reinterpret_cast<const float4 *>(&Bs[cur][kk][tx * 4]);
            const float4 b1 = *reinterpret_cast<const float4 *>(&Bs[cur][kk][64 + tx * 4]);
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
        }
        if (kt + 1 < nk) {
            const int nx = cur ^ 1;
            *reinterpret_cast<float4 *>(&As[nx][ak][ar]) = ra;
            *reinterpret_cast<float4 *>(&Bs[nx][bk][bc]) = rb;
        }
        __syncthreads();
        cur ^= 1;
    }
    // this thread holds atoms ty*4..+3 and 64+ty*4..+3 of the tile: float4 runs along the atom axis
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const int col = n0 + (j < 4 ? tx * 4 + j : 64 + tx * 4 + (j - 4));
        if (col >= N) continue;
        const float bb = EPI == EPI_HIDDEN ? __ldg(bias + col) : 0.f;
#pragma unroll
        for (int ih = 0; ih < 2; ++ih) {
            const int64_t o = ((int64_t)blockIdx.y * N + col) * BM + ih * 64 + ty * 4;
            float4 v = make_float4(acc[ih * 4 + 0][j], acc[ih * 4 + 1][j], acc[ih * 4 + 2][j], acc[ih * 4 + 3][j]);
            if (EPI == EPI_HIDDEN) {
                float4 h, d;
                swish_pair(v.x + bb, h.x, d.x);
                swish_pair(v.y + bb, h.y, d.y);
                swish_pair(v.z + bb, h.z, d.z);
                swish_pair(v.w + bb, h.w, d.w);
                *reinterpret_cast<float4 *>(Ct + o) = h;
                *reinterpret_cast<float4 *>(C2t + o) = d;
            } else if (EPI == EPI_MUL) {
                const float4 dm = __ldg(reinterpret_cast<const float4 *>(Dmult + o));
                v.x *= dm.x; v.y *= dm.y; v.z *= dm.z; v.w *= dm.w;
                *reinterpret_cast<float4 *>(Ct + o) = v;
            } else {
                *reinterpret_cast<float4 *>(Ct + o) = v;
            }
        }
    }
}

static int sgemm(int epi, int64_t M, int N, int K, const float *A, const float *B, float *C, const float *bias,
                 float *C2, const float *Dmul, cudaStream_t st) {
    if (K % BK != 0 || N % 4 != 0) {
        set_error("MLP widths must be multiples of 8 (K = %d) and 4 (N = %d)", K, N);
        return GMNN_UNSUPPORTED;
    }
    dim3 grid((N + BN - 1) / BN, (unsigned)((M + BM - 1) / BM));
    switch (epi) {
        case EPI_PLAIN: k_sgemm<EPI_PLAIN><<<grid, 256, 0, st>>>((int)M, N, K, A, B, N, C, bias, C2, Dmul); break;
        case EPI_HIDDEN: k_sgemm<EPI_HIDDEN><<<grid, 256, 0, st>>>((int)M, N, K, A, B, N, C, bias, C2, Dmul); break;
        default: k_sgemm<EPI_MUL><<<grid, 256, 0, st>>>((int)M, N, K, A, B, N, C, bias, C2, Dmul); break;
    }
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// H tile-transposed (coalesced along atoms): y_m = h . W_last[:, m] + b_last[m]; E^(m) = sigma y_m + mu;
// e_atom = sum_m c_m E^(m).
// Rows row0 .. row0 + rows of one segment (Ht, Wl, bl already point at the segment / its weight set); e_heads and
// e_atom are indexed by the internal atom of the row (row_atom; identity when null).
// One thread per (atom, group of 8 heads): 64 atoms x ceil(M / 8) groups per block, so that a 32-head model spreads
// 8 192 atoms over 128 blocks of 8 warps (one thread per atom for all heads left 64 blocks of 4 warps: 0.54 ms at
// config 4).  Every head's sum runs over k in the same order as before; e_atom = sum_m head_w[m] E^(m) is chained in
// head order by the first group's thread from the energies the groups leave in shared memory.
constexpr int HEADS_ATOMS = 64, HEADS_MAX = 64;
__global__ void __launch_bounds__(HEADS_ATOMS *(HEADS_MAX / 8))
k_heads(int64_t row0, int64_t rows, const float *__restrict__ Ht, int Hd, const float *__restrict__ Wl,
        const float *__restrict__ bl, int M, const float4 *__restrict__ pos4, const float *__restrict__ scale,
        const float *__restrict__ shift, const float *__restrict__ head_w, float *__restrict__ e_heads,
        float *__restrict__ e_atom, const int32_t *__restrict__ row_atom, const float *__restrict__ e_zbl) {
    __shared__ float s_em[HEADS_MAX * HEADS_ATOMS];
    const int a = threadIdx.x % HEADS_ATOMS, g = threadIdx.x / HEADS_ATOMS;
    const int64_t r = blockIdx.x * (int64_t)HEADS_ATOMS + a;
    const bool live = r < rows;
    const int64_t i = live ? (row_atom ? (int64_t)row_atom[row0 + r] : row0 + r) : 0;
    if (live) {
        const float *h = Ht + (r >> 7) * Hd * 128 + (r & 127);  // tile-transposed [rows / 128][Hd][128]
        const int z = __float_as_int(pos4[i].w);
        // ZBL (an empirical correction outside the network): every head's energy carries it once
        const float sg = __ldg(&scale[z]), mu = __ldg(&shift[z]) + (e_zbl ? __ldg(&e_zbl[i]) : 0.f);
        const int m0 = 8 * g;
        float p[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        const int nm = M - m0 < 8 ? M - m0 : 8;
        if (nm == 1) {
#pragma unroll 8
            for (int k = 0; k < Hd; ++k) p[0] = fmaf(__ldg(h + (int64_t)k * 128), __ldg(&Wl[(int64_t)k * M + m0]), p[0]);
        } else {
            for (int k = 0; k < Hd; ++k) {
                const float hv = __ldg(h + (int64_t)k * 128);
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    if (c < nm) p[c] = fmaf(hv, __ldg(&Wl[(int64_t)k * M + m0 + c]), p[c]);
            }
        }
#pragma unroll
        for (int c = 0; c < 8; ++c)
            if (c < nm) {
                const float em = sg * (p[c] + __ldg(&bl[m0 + c])) + mu;
                e_heads[i * (int64_t)M + m0 + c] = em;
                s_em[(m0 + c) * HEADS_ATOMS + a] = em;
            }
    }
    __syncthreads();
    if (live && g == 0) {
        float e = 0.f;
        for (int m = 0; m < M; ++m) e = fmaf(__ldg(&head_w[m]), s_em[m * HEADS_ATOMS + a], e);
        e_atom[i] = e;
    }
}

// v[k] = sum_m c_m W_last[k][m]
__global__ void k_head_vec(int Hd, int M, const float *__restrict__ Wl, const float *__restrict__ c, float *v) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Hd) return;
    float a = 0.f;
    for (int m = 0; m < M; ++m) a = fmaf(__ldg(&c[m]), __ldg(&Wl[(int64_t)k * M + m]), a);
    v[k] = a;
}

// Bv[k][n] = v[k] WT[k][n]
__global__ void k_scale_rows(int rows, int cols, const float *__restrict__ WT, const float *__restrict__ v, float *Bv) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= (int64_t)rows * cols) return;
    Bv[t] = __ldg(&v[t / cols]) * __ldg(&WT[t]);
}

// BvT[n][k] = W[n][k] v[k]
__global__ void k_scale_cols(int rows, int cols, const float *__restrict__ W, const float *__restrict__ v, float *BvT) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= (int64_t)rows * cols) return;
    BvT[t] = __ldg(&v[t % cols]) * __ldg(&W[t]);
}

int launch_mlp_forward_simt(gmnn_system *s, cudaStream_t st) {
    const gmnn_model *m = s->model;
    s->heads_fused = false;
    MlpSeg seg[MAX_SPECIES];
    const int ns = mlp_segments(s, seg);
    const float *X = s->G;
    for (int l = 0; l < m->hp.n_hidden; ++l) {
        const int fi = m->dims[l], fo = m->dims[l + 1];
        for (int q = 0; q < ns; ++q) {
            const int64_t r0 = seg[q].row0;
            int rc = sgemm(EPI_HIDDEN, seg[q].rows, fo, fi, tile_rows(X, r0, fi), m->W[l] + seg[q].set * m->wsize(l),
                           tile_rows(s->H[l], r0, fo), m->b[l] + seg[q].set * fo, tile_rows(s->D[l], r0, fo), nullptr, st);
            if (rc) return rc;
        }
        X = s->H[l];
    }
    return GMNN_OK;
}

// Single head fused into the last GEMM epilogue (mlp_tc.cu): add the partial sums in slot order.
__global__ void k_heads_finish(int64_t row0, int64_t rows, const float *__restrict__ ypart, int n_slots, int64_t m_pad,
                               const float *__restrict__ bl, const float4 *__restrict__ pos4,
                               const float *__restrict__ scale, const float *__restrict__ shift,
                               const float *__restrict__ head_w, float *__restrict__ e_heads, float *__restrict__ e_atom,
                               const int32_t *__restrict__ row_atom, const float *__restrict__ e_zbl) {
    const int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (r >= rows) return;
    float y = 0.f;
    for (int q = 0; q < n_slots; ++q) y += __ldg(ypart + q * m_pad + row0 + r);
    const int64_t i = row_atom ? (int64_t)row_atom[row0 + r] : row0 + r;
    const int z = __float_as_int(pos4[i].w);
    const float em = __ldg(&scale[z]) * (y + __ldg(&bl[0])) + (__ldg(&shift[z]) + (e_zbl ? __ldg(&e_zbl[i]) : 0.f));
    if (e_heads) {
        e_heads[i] = em;
        e_atom[i] = __ldg(&head_w[0]) * em;
    } else {  // folded mean head of a multi-head model (MD): the head's value is the energy
        e_atom[i] = em;
    }
}

int launch_mlp_heads(gmnn_system *s, const float *head_w_dev, cudaStream_t st) {
    const gmnn_model *m = s->model;
    const int L = m->hp.n_hidden, Hd = m->dims[L], M = m->dims[L + 1];
    MlpSeg seg[MAX_SPECIES];
    const int ns = mlp_segments(s, seg);
    if (!s->heads_fused && Hd > 1024) {
        set_error("last hidden width > 1024");
        return GMNN_UNSUPPORTED;
    }
    for (int q = 0; q < ns; ++q) {
        const int64_t r0 = seg[q].row0, real = seg[q].real;
        const int t = seg[q].set;
        if (s->heads_fused) {
            const bool mean = m->hp.n_heads > 1;  // fused on a multi-head model: the folded mean head (use_mean_head)
            k_heads_finish<<<(unsigned)((real + 255) / 256), 256, 0, st>>>(
                r0, real, s->ypart, s->head_slots, (s->n_rows + 127) / 128 * 128,
                mean ? m->w_mean + (size_t)t * (Hd + 1) + Hd : m->b[L] + (size_t)t * M, s->pos4, m->scale, m->shift,
                head_w_dev, mean ? nullptr : s->e_heads, s->e_atom, s->row_atom, s->e_zbl);
        } else {
            k_heads<<<(unsigned)((real + HEADS_ATOMS - 1) / HEADS_ATOMS), HEADS_ATOMS * ((M + 7) / 8), 0, st>>>(
                r0, real, tile_rows(s->H[L - 1], r0, Hd), Hd, m->W[L] + t * m->wsize(L), m->b[L] + (size_t)t * M, M, s->pos4,
                m->scale, m->shift, head_w_dev, s->e_heads, s->e_atom, s->row_atom, s->e_zbl);
        }
        GMNN_LAUNCHED();
    }
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// Seeds the backward for the head weights c (device [n_heads]): vhead = W_last c, Bv = diag(vhead) W^T.
int launch_mlp_seed(gmnn_system *s, const float *head_w_dev, cudaStream_t st) {
    const gmnn_model *m = s->model;
    const int L = m->hp.n_hidden;
    const int Hd = m->dims[L], prev = m->dims[L - 1];
    const size_t bv = (size_t)Hd * prev;
    for (int t = 0; t < m->n_sets; ++t) {  // one seeded operand per weight set
        float *v = s->vhead + (size_t)t * Hd;
        k_head_vec<<<(Hd + 127) / 128, 128, 0, st>>>(Hd, m->dims[L + 1], m->W[L] + t * m->wsize(L), head_w_dev, v);
        GMNN_LAUNCHED();
        if (s->mlp_precision == GMNN_MLP_FP32)
            k_scale_rows<<<(unsigned)((bv + 255) / 256), 256, 0, st>>>(Hd, prev, m->WT[L - 1] + t * bv, v, s->Bv + t * bv);
        else
            k_scale_cols<<<(unsigned)((bv + 255) / 256), 256, 0, st>>>(prev, Hd, m->W[L - 1] + t * bv, v, s->BvT + t * bv);
        GMNN_LAUNCHED();
    }
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_mlp_backward_simt(gmnn_system *s, const float *head_w_dev, cudaStream_t st) {
    const gmnn_model *m = s->model;
    const int L = m->hp.n_hidden;
    int rc = GMNN_OK;
    const bool keep = head_w_dev == m->head_mean_w;  // see launch_mlp_backward_tc
    if (!(keep && s->seed_w == head_w_dev && s->seed_prec == s->mlp_precision)) {
        s->seed_w = nullptr;
        if ((rc = launch_mlp_seed(s, head_w_dev, st))) return rc;
        if (keep) s->seed_w = head_w_dev, s->seed_prec = s->mlp_precision;
    }
    MlpSeg seg[MAX_SPECIES];
    const int ns = mlp_segments(s, seg);
    const float *Aop = s->D[L - 1];
    int cur = 0;
    for (int l = L - 1; l >= 0; --l) {
        // out[rows][dims[l]] = Aop[rows][dims[l+1]] . Bop[dims[l+1]][dims[l]], Bop = diag(v) W^T of the last hidden
        // layer first, then W^T of the layers below
        const int fo = m->dims[l], fi = m->dims[l + 1];
        for (int q = 0; q < ns; ++q) {
            const int64_t r0 = seg[q].row0;
            const float *Bop = (l == L - 1) ? s->Bv + seg[q].set * m->wsize(l) : m->WT[l] + seg[q].set * m->wsize(l);
            if (l > 0)
                rc = sgemm(EPI_MUL, seg[q].rows, fo, fi, tile_rows(Aop, r0, fi), Bop, tile_rows(s->dZ[cur], r0, fo), nullptr,
                           nullptr, tile_rows(s->D[l - 1], r0, fo), st);
            else
                rc = sgemm(EPI_PLAIN, seg[q].rows, fo, fi, tile_rows(Aop, r0, fi), Bop, tile_rows(s->dG, r0, fo), nullptr, nullptr,
                           nullptr, st);
            if (rc) return rc;
        }
        if (l > 0) {
            Aop = s->dZ[cur];
            cur ^= 1;
        }
    }
    return GMNN_OK;
}

}  // namespace gmnn
