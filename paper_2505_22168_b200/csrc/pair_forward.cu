// pair_forward.cu -- a4 + a5: Psi[i][s][m] = sum_j R_s(r_ij) mono_m(u_ij)   (Eq. 2).
// LPA lanes share one centre atom and stride over its neighbour row with 16-byte loads of packed entries; each
// neighbour costs one float4 gather of pos4 (L1/L2 resident: atoms are cell sorted).  The species-pair table beta
// sits in shared memory.  Per-lane partial moment sums (100 registers) are combined by xor shuffles inside the
// lane group.
#include "pair_common.cuh"

namespace gmnn {

// ---------------------------------------------------------------------------------------------
// a4 + a5: pair radial functions and moment accumulation
// ---------------------------------------------------------------------------------------------
template <int NR, int NB, int LPA, bool GENERAL>
__global__ void __launch_bounds__(128)
k_pair_forward(int64_t N, const float4 *__restrict__ pos4, const uint32_t *__restrict__ nbr,
               const int32_t *__restrict__ count, int cap, Geometry geo, RadialParams rp,
               const float *__restrict__ beta, float *__restrict__ psi, const int32_t *__restrict__ mrow,
               float *__restrict__ e_zbl) {
    constexpr int KB = (NB + 3) & ~3;
    constexpr int ROW = NR * KB;  // floats per (zi, zj) block of the table
    extern __shared__ float s_beta[];
    for (int q = threadIdx.x; q < rp.n_species * rp.n_species * ROW; q += blockDim.x) s_beta[q] = beta[q];
    __syncthreads();

    const int64_t gt = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t i = gt / LPA;
    const int sub = (int)(gt % LPA);
    const bool live = i < N;
    // moment sums as float2 pairs (m = 2q, 2q + 1): the accumulation runs on the packed fp32 FMA
    // (FFMA2: same flop rate as FFMA, half the issue slots, and this kernel is issue-bound)
    float2 acc[NR][PSI / 2];
#pragma unroll
    for (int s = 0; s < NR; ++s)
#pragma unroll
        for (int q = 0; q < PSI / 2; ++q) acc[s][q] = make_float2(0.f, 0.f);
    float ez = 0.f;  // ZBL: half of every pair's repulsion, summed over the centre's pairs

    if (live) {
        const float4 xi = pos4[i];
        const int zi = __float_as_int(xi.w);
        const int cnt = count[i];
        const uint4 *row = reinterpret_cast<const uint4 *>(nbr + i * (int64_t)cap);
        // the entries of the NEXT iteration are loaded one iteration ahead: row -> pos4[j] is a chain of two
        // dependent global loads, and this takes the first off the critical path (-12 % at config 5; also
        // prefetching the neighbours' position records into L1 from entries two iterations ahead was slower)
        uint4 e_next = sub * 4 < cnt ? __ldg(&row[sub]) : make_uint4(0u, 0u, 0u, 0u);
        for (int k4 = sub; k4 * 4 < cnt; k4 += LPA) {
            const uint4 e4 = e_next;
            if ((k4 + LPA) * 4 < cnt) e_next = __ldg(&row[k4 + LPA]);
            const uint32_t ent[4] = {e4.x, e4.y, e4.z, e4.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (k4 * 4 + q >= cnt) break;
                const PairGeom pg = pair_geometry(ent[q], xi, pos4, geo);
                if (pg.r2 < rp.r_cut2) {
                    const float rinv = rsqrtf(pg.r2);
                    const float r = pg.r2 * rinv;
                    float phi[NB], fc, dummy;
                    radial_basis<NB, false, GENERAL>(rp, r, rinv, phi, nullptr, fc, dummy);
                    if (GENERAL && rp.zbl_on && pg.r2 < rp.zbl_r_max2) {
                        float e, de;
                        zbl_half<false>(rp, zi, pg.zj, r, rinv, e, de);
                        ez += e;
                    }
                    const float4 *bt = reinterpret_cast<const float4 *>(s_beta + (zi * rp.n_species + pg.zj) * ROW);
                    float R[NR];
#pragma unroll
                    for (int s = 0; s < NR; ++s) {
                        float sum = 0.f;
#pragma unroll
                        for (int kq = 0; kq < KB / 4; ++kq) {
                            const float4 b = bt[s * (KB / 4) + kq];
                            if (4 * kq + 0 < NB) sum = fmaf(b.x, phi[4 * kq + 0], sum);
                            if (4 * kq + 1 < NB) sum = fmaf(b.y, phi[4 * kq + 1], sum);
                            if (4 * kq + 2 < NB) sum = fmaf(b.z, phi[4 * kq + 2], sum);
                            if (4 * kq + 3 < NB) sum = fmaf(b.w, phi[4 * kq + 3], sum);
                        }
                        R[s] = fc * sum;
                    }
                    float mono[PSI];
                    monomials(pg.dx * rinv, pg.dy * rinv, pg.dz * rinv, mono);
#pragma unroll
                    for (int s = 0; s < NR; ++s) {
                        const float2 R2 = make_float2(R[s], R[s]);
#pragma unroll
                        for (int q = 0; q < PSI / 2; ++q)
                            acc[s][q] = __ffma2_rn(R2, make_float2(mono[2 * q], mono[2 * q + 1]), acc[s][q]);
                    }
                }
            }
        }
    }
    // combine the LPA partial sums (all lanes of the warp take part)
#pragma unroll
    for (int o = LPA / 2; o >= 1; o >>= 1)
#pragma unroll
        for (int s = 0; s < NR; ++s)
#pragma unroll
            for (int q = 0; q < PSI / 2; ++q) {
                acc[s][q].x += __shfl_xor_sync(0xffffffffu, acc[s][q].x, o);
                acc[s][q].y += __shfl_xor_sync(0xffffffffu, acc[s][q].y, o);
            }
    if (GENERAL && e_zbl) {
#pragma unroll
        for (int o = LPA / 2; o >= 1; o >>= 1) ez += __shfl_xor_sync(0xffffffffu, ez, o);
        if (live && sub == 0) e_zbl[i] = ez;
    }
    if (live) {
        const int64_t row = mrow ? (int64_t)mrow[i] : i;  // per-species weight sets: rows grouped by species
        float4 *out = reinterpret_cast<float4 *>(psi + row * (int64_t)(NR * PSI));
#pragma unroll
        for (int q = 0; q < NR * PSI / 4; ++q) {
            if (q % LPA == sub) {
                const int s = (4 * q) / PSI, m = ((4 * q) % PSI) / 2;
                out[q] = make_float4(acc[s][m].x, acc[s][m].y, acc[s][m + 1].x, acc[s][m + 1].y);
            }
        }
    }
}

template <int NR, int NB>
static int pair_forward_lpa(gmnn_system *s, cudaStream_t st, int lpa) {
    const gmnn_model *m = s->model;
    const size_t smem = sizeof(float) * m->rp.n_species * m->rp.n_species * NR * m->rp.kb;
    const unsigned grid = nblocks(s->N * lpa, 128);
    const bool general = m->rp.basis_kind != 0 || m->rp.zbl_on;
#define GMNN_PF(L)                                                                                        \
    case L:                                                                                               \
        if (general)                                                                                      \
            k_pair_forward<NR, NB, L, true><<<grid, 128, smem, st>>>(s->N, s->pos4, s->nbr, s->count, s->cap, s->geo, \
                                                                     m->rp, m->beta, s->psi, s->mrow, s->e_zbl); \
        else                                                                                              \
            k_pair_forward<NR, NB, L, false><<<grid, 128, smem, st>>>(s->N, s->pos4, s->nbr, s->count, s->cap, s->geo, \
                                                                      m->rp, m->beta, s->psi, s->mrow, nullptr); \
        break;
    switch (lpa) {
        GMNN_PF(1) GMNN_PF(2) GMNN_PF(4) GMNN_PF(8) GMNN_PF(16) GMNN_PF(32)
        default:
            set_error("lanes_per_atom must be 1, 2, 4, 8, 16 or 32");
            return GMNN_INVALID_ARG;
    }
#undef GMNN_PF
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_pair_forward(gmnn_system *s, cudaStream_t st) {
    const gmnn_model *m = s->model;
    if (m->hp.n_radial == 5 && m->hp.n_basis == 7) return pair_forward_lpa<5, 7>(s, st, pick_lpa(s));
    set_error("pair kernels are instantiated for n_radial = 5, n_basis = 7 only");
    return GMNN_UNSUPPORTED;
}

}  // namespace gmnn
