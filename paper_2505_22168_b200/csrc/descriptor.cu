// descriptor.cu -- the Gaussian-moment descriptor and its adjoint (SURVEY.md 8(a) rows a4-a6,
// a9-a11; Eq. 2 and 3).
//
//   k_pair_forward      Psi[i][s][m] = sum_j R_s(r_ij) mono_m(u_ij)          (a4, a5)
//   k_contract_forward  G[i][0..F)   = invariants of Psi[i]                   (a6)
//   k_contract_backward A[i][s][m]   = dE/dPsi[i][s][m] from dE/dG[i]         (a9)
//   k_pair_backward     F_i = sum_{j in N(i)} (g_ij - g_ji)                   (a10, a11)
//
// Pair kernels: LPA lanes share one centre atom and stride over its neighbour row with 16-byte
// loads of packed entries; each neighbour costs one float4 gather of pos4 (L1/L2 resident: atoms
// are cell sorted).  The species-pair table beta sits in shared memory.  Per-lane partial moment
// sums (100 registers) are combined by xor shuffles inside the lane group.
// Force reduction, two forms, both without atomics, in a fixed summation order, bit-reproducible
// (the full list is symmetric, (i,j,n) <-> (j,i,-n)):
//   pair buffer (GMNN_FORCE_PAIRBUF, what bench.py times): g_ij is evaluated once per directed pair with
//     the centre's own adjoint A_i and stored into the row of j at the slot of the reverse pair (index
//     built with the list, neighbor.cu); k_force_reduce subtracts each atom's received row in slot order;
//   gather form (GMNN_FORCE_GATHER): each centre evaluates both directions itself, g_ij with A_i and
//     g_ji with the neighbour's A_j (a 400-byte read served by L1/L2).
//
// Per-pair polynomial: E gets sum_s R_s(r) p_s(u) from pair (i,j), p_s(u) = sum_m A_i[s][m]
// mono_m(u), so g_ij = dE/dd = (sum_s R'_s p_s) u + (grad_u q - (u.grad_u q) u) / r with
// q(u) = sum_m (sum_s R_s A[s][m]) mono_m(u).
#include <type_traits>
#include <vector>

#include "contraction.cuh"
#include "gmnn_internal.h"
#include "tc_ptx.cuh"

namespace gmnn {

constexpr float PI_F = 3.14159265358979323846f;

// ---------------------------------------------------------------------------------------------
// geometry of one packed neighbour entry
// ---------------------------------------------------------------------------------------------
struct PairGeom {
    float dx, dy, dz, r2;
    int j, zj;
};

__device__ __forceinline__ float image_diff(float xj, float xi, float shift) {
    // keep the large cancellation exact: combine the lattice shift with whichever coordinate it cancels
    return shift > 0.f ? xj + (shift - xi) : (xj + shift) - xi;
}

__device__ __forceinline__ PairGeom pair_geometry(uint32_t entry, const float4 &xi, const float4 *__restrict__ pos4,
                                                  const Geometry &geo) {
    PairGeom g;
    g.j = (int)(entry & NBR_J_MASK);
    const float4 xj = __ldg(&pos4[g.j]);
    g.zj = __float_as_int(xj.w);
    // lattice shift n1 a + n2 b + n3 c of the entry's image (n_x L_x on an orthorhombic cell)
    const float n1 = (float)((int)((entry >> NBR_J_BITS) & 7u) - 4), n2 = (float)((int)((entry >> (NBR_J_BITS + 3)) & 7u) - 4),
                n3 = (float)((int)((entry >> (NBR_J_BITS + 6)) & 7u) - 4);
    const float sx = lattice_shift(geo, 0, n1, n2, n3), sy = lattice_shift(geo, 1, n1, n2, n3), sz = lattice_shift(geo, 2, n1, n2, n3);
    g.dx = image_diff(xj.x, xi.x, sx);
    g.dy = image_diff(xj.y, xi.y, sy);
    g.dz = image_diff(xj.z, xi.z, sz);
    g.r2 = g.dx * g.dx + g.dy * g.dy + g.dz * g.dz;
    return g;
}

// Phi_k(r) = exp(-gamma (r - mu_k)^2), f_c = 1/2 (1 + cos(pi r / r_cut))   (readings R1-R3)
template <int NB, bool WITH_DERIV>
__device__ __forceinline__ void radial_basis(const RadialParams &rp, float r, float *phi, float *dphi, float &fc,
                                             float &dfc) {
    const float t = r * rp.inv_rc;
    if (WITH_DERIV) {
        float sn, cs;
        sincospif(t, &sn, &cs);
        fc = 0.5f + 0.5f * cs;
        dfc = -0.5f * PI_F * rp.inv_rc * sn;
    } else {
        fc = 0.5f + 0.5f * cospif(t);
    }
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        const float d = r - (rp.r_min + (float)k * rp.delta);
        const float p = __expf(-rp.gamma * d * d);
        phi[k] = p;
        if (WITH_DERIV) dphi[k] = -2.f * rp.gamma * d * p;
    }
}

__device__ __forceinline__ void monomials(float x, float y, float z, float *m) {
    m[0] = 1.f;
    m[1] = x; m[2] = y; m[3] = z;
    m[4] = x * x; m[5] = x * y; m[6] = x * z; m[7] = y * y; m[8] = y * z; m[9] = z * z;
    m[10] = m[4] * x; m[11] = m[4] * y; m[12] = m[4] * z; m[13] = m[7] * x; m[14] = m[5] * z;
    m[15] = m[9] * x; m[16] = m[7] * y; m[17] = m[7] * z; m[18] = m[9] * y; m[19] = m[9] * z;
}

// ---------------------------------------------------------------------------------------------
// a4 + a5: pair radial functions and moment accumulation
// ---------------------------------------------------------------------------------------------
template <int NR, int NB, int LPA>
__global__ void __launch_bounds__(128)
k_pair_forward(int64_t N, const float4 *__restrict__ pos4, const uint32_t *__restrict__ nbr,
               const int32_t *__restrict__ count, int cap, Geometry geo, RadialParams rp,
               const float *__restrict__ beta, float *__restrict__ psi, const int32_t *__restrict__ mrow) {
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
                    radial_basis<NB, false>(rp, r, phi, nullptr, fc, dummy);
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

// ---------------------------------------------------------------------------------------------
// a6: invariants.  One thread per atom, Psi row in registers, straight-line FMA code from
// contraction.cuh.  Features leave through a per-warp shared tile (feature-major, padded to 33)
// so that global stores are contiguous runs of one atom's row.
// ---------------------------------------------------------------------------------------------
template <int NR>
struct FeatChunks {
    using F = Feat<NR>;
    // chunk boundaries in feature space: [0, OFF4) [OFF4, OFF5) [OFF5, OFF6) [OFF6, OFF7) [OFF7, N)
    static constexpr int NCH = 5;
    __host__ __device__ static constexpr int begin(int c) {
        return c == 0 ? 0 : c == 1 ? F::OFF4 : c == 2 ? F::OFF5 : c == 3 ? F::OFF6 : c == 4 ? F::OFF7 : F::N;
    }
    __host__ __device__ static constexpr int chunk_of(int f) {
        return f < F::OFF4 ? 0 : f < F::OFF5 ? 1 : f < F::OFF6 ? 2 : f < F::OFF7 ? 3 : 4;
    }
    __host__ __device__ static constexpr int mask(int c) { return c == 0 ? 0x0F : (0x08 << c); }
    __host__ __device__ static constexpr int max_len() {
        int m = 0;
        for (int c = 0; c < NCH; ++c) m = (begin(c + 1) - begin(c)) > m ? (begin(c + 1) - begin(c)) : m;
        return m;
    }
};

constexpr int CW = 33;  // padded warp tile pitch

template <int NR>
__global__ void __launch_bounds__(128)
k_contract_forward(int64_t N, const float *__restrict__ psi, float *__restrict__ Gt, uint32_t *__restrict__ amax) {
    using F = Feat<NR>;
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;  // blockDim.x == 128 == tile
    float P[NR][PSI];
    if (i < N) {
        const float4 *src = reinterpret_cast<const float4 *>(psi + i * (int64_t)(NR * PSI));
#pragma unroll
        for (int q = 0; q < NR * PSI / 4; ++q) {
            const float4 v = __ldg(&src[q]);
            P[(4 * q) / PSI][(4 * q) % PSI] = v.x;
            P[(4 * q + 1) / PSI][(4 * q + 1) % PSI] = v.y;
            P[(4 * q + 2) / PSI][(4 * q + 2) % PSI] = v.z;
            P[(4 * q + 3) / PSI][(4 * q + 3) % PSI] = v.w;
        }
    } else {
#pragma unroll
        for (int s = 0; s < NR; ++s)
#pragma unroll
            for (int m = 0; m < PSI; ++m) P[s][m] = 0.f;
    }
    // G is tile-transposed ([N/128][F][128], the A-operand layout of the MLP): feature f of the 128
    // atoms of this block is one contiguous 512-byte run, so every store below is coalesced.
    float *g = Gt + (int64_t)blockIdx.x * F::N * 128 + threadIdx.x;
    float gmax = 0.f;  // max |G| of the evaluation: the operand scale of the 3xFP16 MLP (mlp_tc.cu)
    contract_forward<NR>([&](int s, int m) { return P[s][m]; }, [&](int f, float v) {
        g[(int64_t)f * 128] = v;
        gmax = fmaxf(gmax, fabsf(v));
    });
    if (amax) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, o));
        if ((threadIdx.x & 31) == 0 && gmax > 0.f) atomicMax(amax, __float_as_uint(gmax));
    }
}

// ---------------------------------------------------------------------------------------------
// a9: adjoint of the invariants.  One thread per atom, one block per 128-atom tile of dE/dG, which
// the MLP backward writes tile-transposed ([N/128][F][128]): every chunk of feature blocks is one
// contiguous run, brought into shared memory by 1-D bulk copies (cp.async.bulk + mbarrier) into two
// slots so that the next chunk lands while the current one is consumed; reads sG[f][tid] are
// conflict-free.  Psi row and the 100 adjoints live in registers (straight-line FMA code).
// dE/dG arrives without the sigma_Z factor of Eq. 4 (the MLP backward is linear in it); it is
// applied here.
// ---------------------------------------------------------------------------------------------
// c_rot[r][f]: the feature whose channel tuple is that of feature f with every channel shifted by r
// (mod 5): what the representative-tuple code of contract_backward<.., ORBIT = true> reads in round r.
__constant__ uint16_t c_rot[5 * Feat<5>::N];

static int upload_rot_table() {
    using F = Feat<5>;
    constexpr int NR = 5;
    static bool done_on[MAX_DEVICES] = {};  // c_rot is per-device memory
    bool &done = done_on[current_device()];
    if (done) return GMNN_OK;
    std::vector<uint16_t> t((size_t)NR * F::N, 0);
    auto sort2 = [](int &a, int &b) { if (a > b) { int x = a; a = b; b = x; } };
    for (int r = 0; r < NR; ++r) {
        uint16_t *row = t.data() + (size_t)r * F::N;
        auto sh = [&](int x) { return (x + r) % NR; };
        for (int x = 0; x < NR; ++x) row[F::OFF0 + x] = (uint16_t)(F::OFF0 + sh(x));
        for (int s1 = 0; s1 < NR; ++s1)
            for (int s2 = s1; s2 < NR; ++s2) {
                int a = sh(s1), b = sh(s2);
                sort2(a, b);
                row[F::OFF1 + F::pidx(s1, s2)] = (uint16_t)(F::OFF1 + F::pidx(a, b));
                row[F::OFF2 + F::pidx(s1, s2)] = (uint16_t)(F::OFF2 + F::pidx(a, b));
                row[F::OFF3 + F::pidx(s1, s2)] = (uint16_t)(F::OFF3 + F::pidx(a, b));
                for (int s3 = 0; s3 < NR; ++s3) {
                    row[F::OFF5 + F::pidx(s1, s2) * NR + s3] = (uint16_t)(F::OFF5 + F::pidx(a, b) * NR + sh(s3));
                    row[F::OFF6 + F::pidx(s1, s2) * NR + s3] = (uint16_t)(F::OFF6 + F::pidx(a, b) * NR + sh(s3));
                }
                for (int s3 = s2; s3 < NR; ++s3) {
                    int x = sh(s1), y = sh(s2), z = sh(s3);
                    sort2(x, y); sort2(y, z); sort2(x, y);
                    row[F::OFF4 + F::tidx(s1, s2, s3)] = (uint16_t)(F::OFF4 + F::tidx(x, y, z));
                }
            }
        for (int s1 = 0; s1 < NR; ++s1)
            for (int s2 = 0; s2 < NR; ++s2)
                for (int s3 = 0; s3 < NR; ++s3)
                    row[F::OFF7 + (s1 * NR + s2) * NR + s3] = (uint16_t)(F::OFF7 + (sh(s1) * NR + sh(s2)) * NR + sh(s3));
    }
    GMNN_CUDA(cudaMemcpyToSymbol(c_rot, t.data(), t.size() * sizeof(uint16_t)));
    done = true;
    return GMNN_OK;
}

template <int NR>
struct CbSmem {  // shared-memory plan of k_contract_backward, in floats
    using CH = FeatChunks<NR>;
    static constexpr int TB = 128;  // atoms per block = one dG tile
    static constexpr int len(int c) { return CH::begin(c + 1) - CH::begin(c); }
    static constexpr int cmax(int a, int b) { return a > b ? a : b; }
    // slot X: chunk 4 (block 7), then chunks 1 and 3 back to back, then the output transpose
    static constexpr int X = cmax(cmax(len(4), len(1) + len(3)) * TB, 4 * NR * PSI * CW);
    // slot Y: chunk 0, then chunk 2
    static constexpr int Y = cmax(len(0), len(2)) * TB;
    static constexpr size_t bytes(int halves) { return sizeof(float) * (X + Y) * halves + 16 * halves; }
};

// HALVES = 2: one 256-thread block per SM works on two tiles in lock step (the block-wide barriers
// between chunks keep all eight warps inside the same stretch of the ~12 k-instruction straight-line
// body, so they share its instruction-cache lines); HALVES = 1: two independent 128-thread blocks per SM.
// ORBIT: the straight-line body holds only the representative channel tuples (contraction.cuh) and runs
// NR times per chunk, the Psi rows and the adjoints moved down one channel (register moves) after each
// round and the features read through c_rot: a fifth of the code, and each chunk's loop then fits
// the 32 KB instruction cache level for four of its five rounds (the full body is ~170 KB, fetched from
// L2 once per block: ncu shows the no_instruction stalls at every 256-byte boundary).
template <int NR, int HALVES, bool LOCKSTEP, bool ORBIT>
__global__ void __launch_bounds__(128 * HALVES, 3 - HALVES)
k_contract_backward(int64_t N, const float *__restrict__ psi, const float *__restrict__ dGt,
                    const float4 *__restrict__ pos4, const float *__restrict__ scale, float *__restrict__ A,
                    const int32_t *__restrict__ row_atom) {
    using F = Feat<NR>;
    using CH = FeatChunks<NR>;
    using SM = CbSmem<NR>;
    constexpr int TB = SM::TB;
    extern __shared__ __align__(128) float s_cb[];
    const int hf = threadIdx.x >> 7;  // which tile of the block
    float *sX = s_cb + hf * (SM::X + SM::Y), *sY = sX + SM::X;
    const uint32_t barX = tc::smem_u32(s_cb + HALVES * (SM::X + SM::Y)) + 16 * hf, barY = barX + 8;
    const int tid = threadIdx.x & 127, lane = tid & 31, wid = tid >> 5;
    const int64_t tile = blockIdx.x * (int64_t)HALVES + hf;
    const bool active = tile * TB < N;  // the last block of an odd tile count has an idle half
    const int64_t i = tile * TB + tid;
    const float *gt = dGt + tile * (int64_t)(F::N * TB);  // this half's [F][128] tile
    auto issue = [&](float *dst, int c, uint32_t bar) {
        tc::bulk_load_1d(tc::smem_u32(dst), gt + CH::begin(c) * TB, (uint32_t)(SM::len(c) * TB * 4), bar);
    };
    if (tid == 0 && active) {
        tc::mbar_init(barX, 1);
        tc::mbar_init(barY, 1);
        tc::fence_barrier_init();
        tc::mbar_arrive_expect_tx(barY, (uint32_t)(SM::len(0) * TB * 4));
        issue(sY, 0, barY);
        tc::mbar_arrive_expect_tx(barX, (uint32_t)(SM::len(4) * TB * 4));
        issue(sX, 4, barX);
    }
    float P[NR][PSI];
    float sig = 0.f;
    if (i < N) {
        const float4 *src = reinterpret_cast<const float4 *>(psi + i * (int64_t)(NR * PSI));
#pragma unroll
        for (int q = 0; q < NR * PSI / 4; ++q) {
            const float4 v = __ldg(&src[q]);
            P[(4 * q) / PSI][(4 * q) % PSI] = v.x;
            P[(4 * q + 1) / PSI][(4 * q + 1) % PSI] = v.y;
            P[(4 * q + 2) / PSI][(4 * q + 2) % PSI] = v.z;
            P[(4 * q + 3) / PSI][(4 * q + 3) % PSI] = v.w;
        }
        const int64_t atom = row_atom ? (int64_t)row_atom[i] : i;  // N counts rows; padding rows have no atom
        sig = atom >= 0 ? __ldg(&scale[__float_as_int(pos4[atom].w)]) : 0.f;
    } else {
#pragma unroll
        for (int s = 0; s < NR; ++s)
#pragma unroll
            for (int m = 0; m < PSI; ++m) P[s][m] = 0.f;
    }
    float acc[NR][PSI];
#pragma unroll
    for (int s = 0; s < NR; ++s)
#pragma unroll
        for (int m = 0; m < PSI; ++m) acc[s][m] = 0.f;
    __syncthreads();  // barrier initialisation visible to every waiter

    auto run_chunk = [&](auto chunk_tag, const float *buf) {
        constexpr int C = decltype(chunk_tag)::value;
        if constexpr (ORBIT) {
#pragma unroll 1
            for (int r = 0; r < NR; ++r) {
                const uint16_t *rot = c_rot + r * F::N;
                contract_backward<NR, CH::mask(C), true>(
                    [&](int s, int m) { return P[s][m]; },
                    [&](int f) { return buf[((int)rot[f] - CH::begin(C)) * TB + tid]; },
                    [&](int s, int m, float v) { acc[s][m] += v; },
                    [&]() {
                        if (LOCKSTEP) __syncthreads();
                    });
                // static channel s now stands for channel s + r + 1 (after NR rounds: back in place)
#pragma unroll
                for (int m = 0; m < PSI; ++m) {
                    const float p0 = P[0][m], a0 = acc[0][m];
#pragma unroll
                    for (int s = 0; s + 1 < NR; ++s) P[s][m] = P[s + 1][m], acc[s][m] = acc[s + 1][m];
                    P[NR - 1][m] = p0, acc[NR - 1][m] = a0;
                }
            }
        } else {
            contract_backward<NR, CH::mask(C)>(
                [&](int s, int m) { return P[s][m]; },
                [&](int f) { return buf[(f - CH::begin(C)) * TB + tid]; },
                [&](int s, int m, float v) { acc[s][m] += v; },
                [&]() {  // keep the warps of the block in the same stretch of the instruction stream
                    if (LOCKSTEP) __syncthreads();
                });
        }
    };
    if (active) tc::mbar_wait(barY, 0);
    run_chunk(std::integral_constant<int, 0>{}, sY);
    __syncthreads();
    if (tid == 0 && active) {
        tc::fence_proxy_async_smem();
        tc::mbar_arrive_expect_tx(barY, (uint32_t)(SM::len(2) * TB * 4));
        issue(sY, 2, barY);
    }
    if (active) tc::mbar_wait(barX, 0);
    run_chunk(std::integral_constant<int, 4>{}, sX);
    __syncthreads();
    if (tid == 0 && active) {
        tc::fence_proxy_async_smem();
        tc::mbar_arrive_expect_tx(barX, (uint32_t)((SM::len(1) + SM::len(3)) * TB * 4));
        issue(sX, 1, barX);
        issue(sX + SM::len(1) * TB, 3, barX);
    }
    if (active) tc::mbar_wait(barY, 1);
    run_chunk(std::integral_constant<int, 2>{}, sY);
    if (active) tc::mbar_wait(barX, 1);
    run_chunk(std::integral_constant<int, 1>{}, sX);
    run_chunk(std::integral_constant<int, 3>{}, sX + SM::len(1) * TB);
    __syncthreads();

    // transpose the adjoints through slot X (per-warp [NR*PSI][33] tiles) for contiguous row stores
    float *sP = sX + wid * (NR * PSI * CW);
#pragma unroll
    for (int s = 0; s < NR; ++s)
#pragma unroll
        for (int m = 0; m < PSI; ++m) sP[(s * PSI + m) * CW + lane] = sig * acc[s][m];
    __syncwarp();
    const int64_t i0 = i - lane;
    for (int a = 0; a < 32; ++a) {
        const int64_t ia = i0 + a;
        if (ia >= N) break;
        float *dst = A + ia * (int64_t)(NR * PSI);
        for (int q = lane; q < NR * PSI; q += 32) dst[q] = sP[q * CW + a];
    }
}

// ---------------------------------------------------------------------------------------------
// a10 + a11: pair gradient in both directions and the force sum of the centre atom
// ---------------------------------------------------------------------------------------------
// g = dE/dd for one direction.  a(s, q) returns the float4 {A[s][4q..4q+3]}; (x, y, z) is the unit
// vector the centre's polynomial is evaluated at: +u for the centre itself, -u for its neighbour.
template <int NR, class AGet>
__device__ __forceinline__ void pair_gradient(AGet a, const float *R, const float *dR, const float *mono, float x,
                                              float y, float z, float rinv, float &gx, float &gy, float &gz) {
    // mono = monomials of (x, y, z), the direction the polynomial is evaluated at (+u or -u).
    // Both 100-term sums run on the packed fp32 FMA (FFMA2), two monomials per instruction.
    float2 t2[PSI / 2];
#pragma unroll
    for (int q = 0; q < PSI / 2; ++q) t2[q] = make_float2(0.f, 0.f);
    float radial = 0.f;
#pragma unroll
    for (int s = 0; s < NR; ++s) {
        float2 p2 = make_float2(0.f, 0.f);  // p_s(u) = sum_m A[s][m] mono_m, in two partial sums
        const float2 R2 = make_float2(R[s], R[s]);
#pragma unroll
        for (int q = 0; q < PSI / 4; ++q) {
            const float4 v = a(s, q);
            const float2 a01 = make_float2(v.x, v.y), a23 = make_float2(v.z, v.w);
            p2 = __ffma2_rn(a01, make_float2(mono[4 * q], mono[4 * q + 1]), p2);
            p2 = __ffma2_rn(a23, make_float2(mono[4 * q + 2], mono[4 * q + 3]), p2);
            t2[2 * q] = __ffma2_rn(R2, a01, t2[2 * q]);
            t2[2 * q + 1] = __ffma2_rn(R2, a23, t2[2 * q + 1]);
        }
        radial = fmaf(dR[s], p2.x + p2.y, radial);
    }
    float t[PSI];
#pragma unroll
    for (int q = 0; q < PSI / 2; ++q) t[2 * q] = t2[q].x, t[2 * q + 1] = t2[q].y;
    const float xx = mono[4], xy = mono[5], xz = mono[6], yy = mono[7], yz = mono[8], zz = mono[9];
    // grad_u q(u), q = sum_m t_m mono_m
    float wx = t[1] + 2.f * t[4] * x + t[5] * y + t[6] * z + 3.f * t[10] * xx + 2.f * t[11] * xy + 2.f * t[12] * xz +
               t[13] * yy + t[14] * yz + t[15] * zz;
    float wy = t[2] + t[5] * x + 2.f * t[7] * y + t[8] * z + t[11] * xx + 2.f * t[13] * xy + t[14] * xz +
               3.f * t[16] * yy + 2.f * t[17] * yz + t[18] * zz;
    float wz = t[3] + t[6] * x + t[8] * y + 2.f * t[9] * z + t[12] * xx + t[14] * xy + 2.f * t[15] * xz + t[17] * yy +
               2.f * t[18] * yz + 3.f * t[19] * zz;
    const float wu = wx * x + wy * y + wz * z;
    gx = radial * x + (wx - wu * x) * rinv;
    gy = radial * y + (wy - wu * y) * rinv;
    gz = radial * z + (wz - wu * z) * rinv;
}

// PAIRBUF = false: gather form, both directions per entry, F_i complete.
// PAIRBUF = true : own direction only; g_ij goes to gbuf[j][rev] (the slot of (i, -n) in the row of
//                  j), f_int gets sum_j g_ij, and k_force_reduce subtracts the received row.
// VIRIAL: also leaves vir_atom[c][i] = -sum_j d_a g_b (c = 3 a + b) over the centre's own directed pairs, whose sum
// over the atoms is the virial W = -sum_pairs d (x) g = -dE/d strain (oracle O-16).
template <int NR, int NB, int LPA, bool PAIRBUF, bool VIRIAL>
__global__ void __launch_bounds__(128)
k_pair_backward(int64_t N, const float4 *__restrict__ pos4, const uint32_t *__restrict__ nbr,
                const int32_t *__restrict__ count, int cap, Geometry geo, RadialParams rp,
                const float *__restrict__ beta, const float *__restrict__ A, float *__restrict__ f_int,
                const uint16_t *__restrict__ rev, float4 *__restrict__ gbuf, const int32_t *__restrict__ mrow,
                float *__restrict__ vir_atom) {
    constexpr int KB = (NB + 3) & ~3;
    constexpr int ROW = NR * KB;
    constexpr int GROUPS = 128 / LPA;
    extern __shared__ float s_mem[];
    float *s_beta = s_mem;
    float4 *s_A = reinterpret_cast<float4 *>(s_mem + ((rp.n_species * rp.n_species * ROW + 3) & ~3));
    for (int q = threadIdx.x; q < rp.n_species * rp.n_species * ROW; q += blockDim.x) s_beta[q] = beta[q];
    const int64_t gt = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t i = gt / LPA;
    const int sub = (int)(gt % LPA);
    const int grp = threadIdx.x / LPA;
    const bool live = i < N;
    // stage A_i of the block's centres: GROUPS rows of NR*PSI/4 float4
    {
        const int64_t first = blockIdx.x * (int64_t)GROUPS;
        const float4 *src = reinterpret_cast<const float4 *>(A);
        for (int q = threadIdx.x; q < GROUPS * (NR * PSI / 4); q += blockDim.x) {
            const int64_t ia = first + q / (NR * PSI / 4);
            const int64_t ra = (mrow && ia < N) ? (int64_t)mrow[ia] : ia;  // row of the adjoint (species-grouped rows)
            s_A[q] = ia < N ? __ldg(&src[ra * (NR * PSI / 4) + q % (NR * PSI / 4)]) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    __syncthreads();
    float fx = 0.f, fy = 0.f, fz = 0.f;
    float vir[VIRIAL ? 9 : 1];
#pragma unroll
    for (int c = 0; c < (VIRIAL ? 9 : 1); ++c) vir[c] = 0.f;
    if (live) {
        const float4 xi = pos4[i];
        const int zi = __float_as_int(xi.w);
        const int cnt = count[i];
        const uint4 *row = reinterpret_cast<const uint4 *>(nbr + i * (int64_t)cap);
        const float4 *Ai = s_A + grp * (NR * PSI / 4);
        const uint2 *rrow = reinterpret_cast<const uint2 *>(rev + (PAIRBUF ? i * (int64_t)cap : 0));
        // entries (and reverse slots) of the next iteration are loaded one iteration ahead (see k_pair_forward)
        uint4 e_next = make_uint4(0u, 0u, 0u, 0u);
        uint2 r_next = make_uint2(0u, 0u);
        if (sub * 4 < cnt) {
            e_next = __ldg(&row[sub]);
            if (PAIRBUF) r_next = __ldg(&rrow[sub]);
        }
        for (int k4 = sub; k4 * 4 < cnt; k4 += LPA) {
            const uint4 e4 = e_next;
            const uint2 r2 = r_next;
            if ((k4 + LPA) * 4 < cnt) {
                e_next = __ldg(&row[k4 + LPA]);
                if (PAIRBUF) r_next = __ldg(&rrow[k4 + LPA]);
            }
            const uint32_t ent[4] = {e4.x, e4.y, e4.z, e4.w};
            uint32_t rv[4] = {0u, 0u, 0u, 0u};
            if (PAIRBUF) rv[0] = r2.x & 0xFFFFu, rv[1] = r2.x >> 16, rv[2] = r2.y & 0xFFFFu, rv[3] = r2.y >> 16;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (k4 * 4 + q >= cnt) break;
                const PairGeom pg = pair_geometry(ent[q], xi, pos4, geo);
                if (PAIRBUF && rv[q] == 0xFFFFu) continue;  // no partner (overflowed rebuild): flagged by k_build_rev
                float4 *slot = PAIRBUF ? gbuf + (int64_t)pg.j * cap + rv[q] : nullptr;
                if (PAIRBUF && pg.r2 >= rp.r_cut2) *slot = make_float4(0.f, 0.f, 0.f, 0.f);  // skin shell
                if (pg.r2 < rp.r_cut2) {
                    const float rinv = rsqrtf(pg.r2);
                    const float r = pg.r2 * rinv;
                    float phi[NB], dphi[NB], fc, dfc;
                    radial_basis<NB, true>(rp, r, phi, dphi, fc, dfc);
                    const float ux = pg.dx * rinv, uy = pg.dy * rinv, uz = pg.dz * rinv;
                    float mono[PSI];
                    monomials(ux, uy, uz, mono);
                    float gxo, gyo, gzo, gxr = 0.f, gyr = 0.f, gzr = 0.f;
#pragma unroll
                    for (int dir = 0; dir < (PAIRBUF ? 1 : 2); ++dir) {
                        // dir 0: centre i, table beta[zi][zj], adjoint A_i, direction +u
                        // dir 1: centre j, table beta[zj][zi], adjoint A_j, direction -u
                        const int za = dir == 0 ? zi : pg.zj, zb = dir == 0 ? pg.zj : zi;
                        const float4 *bt = reinterpret_cast<const float4 *>(s_beta + (za * rp.n_species + zb) * ROW);
                        float R[NR], dR[NR];
#pragma unroll
                        for (int s = 0; s < NR; ++s) {
                            float2 sd = make_float2(0.f, 0.f);  // (sum beta phi, sum beta phi'): one FFMA2 per term
#pragma unroll
                            for (int kq = 0; kq < KB / 4; ++kq) {
                                const float4 b = bt[s * (KB / 4) + kq];
                                const float bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
                                for (int c = 0; c < 4; ++c)
                                    if (4 * kq + c < NB)
                                        sd = __ffma2_rn(make_float2(bv[c], bv[c]), make_float2(phi[4 * kq + c], dphi[4 * kq + c]), sd);
                            }
                            R[s] = fc * sd.x;
                            dR[s] = dfc * sd.x + fc * sd.y;
                        }
                        if (dir == 0) {
                            pair_gradient<NR>([&](int s, int qq) { return Ai[s * (PSI / 4) + qq]; }, R, dR, mono, ux, uy,
                                              uz, rinv, gxo, gyo, gzo);
                        } else {
                            const float4 *Aj = reinterpret_cast<const float4 *>(A) +
                                               (int64_t)(mrow ? mrow[pg.j] : pg.j) * (NR * PSI / 4);
                            float mono_r[PSI];  // the neighbour sees the bond reversed
                            monomials(-ux, -uy, -uz, mono_r);
                            float hx, hy, hz;  // gradient with respect to (-u): g_ji in the frame of d_ji = -d_ij
                            pair_gradient<NR>([&](int s, int qq) { return __ldg(&Aj[s * (PSI / 4) + qq]); }, R, dR, mono_r,
                                              -ux, -uy, -uz, rinv, hx, hy, hz);
                            gxr = hx, gyr = hy, gzr = hz;
                        }
                    }
                    if (PAIRBUF) *slot = make_float4(gxo, gyo, gzo, 0.f);
                    if (VIRIAL) {
                        const float dv[3] = {pg.dx, pg.dy, pg.dz}, gv[3] = {gxo, gyo, gzo};
#pragma unroll
                        for (int a = 0; a < 3; ++a)
#pragma unroll
                            for (int b = 0; b < 3; ++b) vir[3 * a + b] = fmaf(-dv[a], gv[b], vir[3 * a + b]);
                    }
                    // F_i += g_ij - g_ji   (g_ji = dE_j/dd_ji, d_ji = -d_ij)
                    fx += gxo - gxr;
                    fy += gyo - gyr;
                    fz += gzo - gzr;
                }
            }
        }
    }
#pragma unroll
    for (int o = LPA / 2; o >= 1; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o);
        fy += __shfl_xor_sync(0xffffffffu, fy, o);
        fz += __shfl_xor_sync(0xffffffffu, fz, o);
    }
    if (live && sub == 0) {
        f_int[3 * i] = fx;
        f_int[3 * i + 1] = fy;
        f_int[3 * i + 2] = fz;
    }
    if (VIRIAL) {
#pragma unroll
        for (int c = 0; c < 9; ++c) {
#pragma unroll
            for (int o = LPA / 2; o >= 1; o >>= 1) vir[c] += __shfl_xor_sync(0xffffffffu, vir[c], o);
            if (live && sub == 0) vir_atom[(int64_t)c * N + i] = vir[c];
        }
    }
}

// a11 (pair-buffer form): F_i = sum_j g_ij (already in f_int) - sum_k gbuf[i][k], the g_ji received
// from the neighbours, summed in slot order by LPA lanes (fixed order: bit-reproducible).
template <int LPA>
__global__ void __launch_bounds__(256)
k_force_reduce(int64_t N, const int32_t *__restrict__ count, int cap, const float4 *__restrict__ gbuf,
               float *__restrict__ f_int) {
    const int64_t gt = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t i = gt / LPA;
    const int sub = (int)(gt % LPA);
    float fx = 0.f, fy = 0.f, fz = 0.f;
    if (i < N) {
        const int cnt = count[i];
        const float4 *row = gbuf + i * (int64_t)cap;
        for (int k = sub; k < cnt; k += LPA) {
            const float4 g = __ldcs(&row[k]);
            fx += g.x, fy += g.y, fz += g.z;
        }
    }
#pragma unroll
    for (int o = LPA / 2; o >= 1; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o);
        fy += __shfl_xor_sync(0xffffffffu, fy, o);
        fz += __shfl_xor_sync(0xffffffffu, fz, o);
    }
    if (i < N && sub == 0) {
        f_int[3 * i] -= fx;
        f_int[3 * i + 1] -= fy;
        f_int[3 * i + 2] -= fz;
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static inline unsigned nblocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }

static int pick_lpa(const gmnn_system *s) {
    if (s->lanes_per_atom > 0) return s->lanes_per_atom;
    // enough warps to fill 148 SMs several times over: small systems spread one atom over more lanes
    if (s->N >= 262144) return 2;  // measured at 524 288 atoms: 2 beats 4 by 5 % in both pair kernels
    if (s->N >= 65536) return 4;
    if (s->N >= 8192) return 8;
    return 32;
}

template <int NR, int NB>
static int pair_forward_lpa(gmnn_system *s, cudaStream_t st, int lpa) {
    const gmnn_model *m = s->model;
    const size_t smem = sizeof(float) * m->rp.n_species * m->rp.n_species * NR * m->rp.kb;
    const unsigned grid = nblocks(s->N * lpa, 128);
#define GMNN_PF(L)                                                                                        \
    case L:                                                                                               \
        k_pair_forward<NR, NB, L><<<grid, 128, smem, st>>>(s->N, s->pos4, s->nbr, s->count, s->cap, s->geo, \
                                                           m->rp, m->beta, s->psi, s->mrow);              \
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

template <int NR, int NB>
static int pair_backward_lpa(gmnn_system *s, cudaStream_t st, int lpa) {
    const gmnn_model *m = s->model;
    const int beta_floats = (m->rp.n_species * m->rp.n_species * NR * m->rp.kb + 3) & ~3;
    const size_t smem = sizeof(float) * (beta_floats + (128 / lpa) * NR * PSI);
    const unsigned grid = nblocks(s->N * lpa, 128);
    const bool pairbuf = s->force_mode == GMNN_FORCE_PAIRBUF;
    const bool virial = s->want_virial && s->vir_atom != nullptr;
    if (pairbuf && !(s->list_has_rev && s->rev && s->gbuf)) {
        set_error("force_mode changed after the list was built: call gmnn_build_neighbors again");
        return GMNN_INVALID_ARG;
    }
#define GMNN_PB_LAUNCH(L, PB, VIR)                                                                         \
    k_pair_backward<NR, NB, L, PB, VIR><<<grid, 128, smem, st>>>(s->N, s->pos4, s->nbr, s->count, s->cap, s->geo, m->rp, \
                                                                m->beta, s->A, s->f_int, PB ? s->rev : nullptr, \
                                                                PB ? s->gbuf : nullptr, s->mrow, VIR ? s->vir_atom : nullptr)
#define GMNN_PB(L)                                                                                         \
    case L: {                                                                                              \
        static size_t opted_on[MAX_DEVICES] = {};                                                          \
        size_t &opted = opted_on[current_device()];                                                        \
        if (smem > 48 * 1024 && smem > opted) {                                                            \
            GMNN_CUDA(cudaFuncSetAttribute(k_pair_backward<NR, NB, L, false, false>,                       \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));       \
            GMNN_CUDA(cudaFuncSetAttribute(k_pair_backward<NR, NB, L, true, false>,                        \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));       \
            GMNN_CUDA(cudaFuncSetAttribute(k_pair_backward<NR, NB, L, false, true>,                        \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));       \
            GMNN_CUDA(cudaFuncSetAttribute(k_pair_backward<NR, NB, L, true, true>,                         \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));       \
            opted = smem;                                                                                  \
        }                                                                                                  \
        if (pairbuf && virial) GMNN_PB_LAUNCH(L, true, true);                                              \
        else if (pairbuf) GMNN_PB_LAUNCH(L, true, false);                                                  \
        else if (virial) GMNN_PB_LAUNCH(L, false, true);                                                   \
        else GMNN_PB_LAUNCH(L, false, false);                                                              \
    } break;
    switch (lpa) {
        GMNN_PB(1) GMNN_PB(2) GMNN_PB(4) GMNN_PB(8) GMNN_PB(16) GMNN_PB(32)
        default:
            set_error("lanes_per_atom must be 1, 2, 4, 8, 16 or 32");
            return GMNN_INVALID_ARG;
    }
#undef GMNN_PB
#undef GMNN_PB_LAUNCH
    GMNN_LAUNCHED();
    if (pairbuf) {
        k_force_reduce<8><<<nblocks(s->N * 8, 256), 256, 0, st>>>(s->N, s->count, s->cap, s->gbuf, s->f_int);
        GMNN_LAUNCHED();
    }
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_pair_forward(gmnn_system *s, cudaStream_t st) {
    const gmnn_model *m = s->model;
    if (m->hp.n_radial == 5 && m->hp.n_basis == 7) return pair_forward_lpa<5, 7>(s, st, pick_lpa(s));
    set_error("pair kernels are instantiated for n_radial = 5, n_basis = 7 only");
    return GMNN_UNSUPPORTED;
}

int launch_pair_backward(gmnn_system *s, cudaStream_t st) {
    const gmnn_model *m = s->model;
    if (m->hp.n_radial == 5 && m->hp.n_basis == 7) return pair_backward_lpa<5, 7>(s, st, pick_lpa(s));
    set_error("pair kernels are instantiated for n_radial = 5, n_basis = 7 only");
    return GMNN_UNSUPPORTED;
}

int launch_contract_forward(gmnn_system *s, cudaStream_t st) {
    constexpr int NR = 5;
    k_contract_forward<NR><<<nblocks(s->n_rows, 128), 128, 0, st>>>(s->n_rows, s->psi, s->G,
                                                               s->mlp_precision == GMNN_MLP_3XF16 ? s->amax + AMAX_G : nullptr);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// The shipped kernel is k_contract_backward<NR, 1, false, true>: one tile per block, orbit-representative
// body.  The superseded shapes (two tiles per block, lock-step barriers, the fully unrolled body: config 5
// 2.57 / 2.25 / 1.23 ms against 1.02 ms) are instantiated only in -DGMNN_EXPERIMENTS builds, behind the
// knob "cb_halves" (1..6).
#ifdef GMNN_EXPERIMENTS
int g_cb_halves = 6;
#endif

template <int NR, int HALVES, bool LOCKSTEP, bool ORBIT>
static int launch_cb(gmnn_system *s, cudaStream_t st) {
    static bool attr_on[MAX_DEVICES] = {};
    bool &attr_set = attr_on[current_device()];
    if (!attr_set) {
        GMNN_CUDA(cudaFuncSetAttribute(k_contract_backward<NR, HALVES, LOCKSTEP, ORBIT>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CbSmem<NR>::bytes(HALVES)));
        attr_set = true;
    }
    const unsigned tiles = nblocks(s->n_rows, 128);
    k_contract_backward<NR, HALVES, LOCKSTEP, ORBIT><<<(tiles + HALVES - 1) / HALVES, 128 * HALVES, CbSmem<NR>::bytes(HALVES), st>>>(
        s->n_rows, s->psi, s->dG, s->pos4, s->model->scale, s->A, s->row_atom);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_contract_backward(gmnn_system *s, cudaStream_t st) {
    constexpr int NR = 5;
    int rc;
    if ((rc = upload_rot_table())) return rc;
#ifdef GMNN_EXPERIMENTS
    switch (g_cb_halves) {
        case 1: return launch_cb<NR, 1, false, false>(s, st);
        case 2: return launch_cb<NR, 2, true, false>(s, st);
        case 3: return launch_cb<NR, 1, true, false>(s, st);
        case 4: return launch_cb<NR, 2, true, true>(s, st);
        case 5: return launch_cb<NR, 1, true, true>(s, st);
        default: break;
    }
#endif
    return launch_cb<NR, 1, false, true>(s, st);
}

}  // namespace gmnn
