// descriptor.cu -- the invariants of the Gaussian-moment descriptor and their adjoint (
// PAPER.md:54-61, Eq. 3).  The pair kernels around them are pair_forward.cu / pair_backward.cu.
//
//   k_contract_forward  G[i][0..F)   = invariants of Psi[i]                   (a6)
//   k_contract_backward A[i][s][m]   = dE/dPsi[i][s][m] from dE/dG[i]         (a9)
#include <type_traits>
#include <vector>

#include "contraction.cuh"
#include "gmnn_internal.h"
#include "tc_ptx.cuh"

namespace gmnn {

static inline unsigned nblocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }

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
                    const int32_t *__restrict__ row_atom, int heads) {
    using F = Feat<NR>;
    using CH = FeatChunks<NR>;
    using SM = CbSmem<NR>;
    constexpr int TB = SM::TB;
    extern __shared__ __align__(128) float s_cb[];
    const int hf = threadIdx.x >> 7;  // which tile of the block
    float *sX = s_cb + hf * (SM::X + SM::Y), *sY = sX + SM::X;
    const uint32_t barX = tc::smem_u32(s_cb + HALVES * (SM::X + SM::Y)) + 16 * hf, barY = barX + 8;
    const int tid = threadIdx.x & 127, lane = tid & 31, wid = tid >> 5;
    // heads > 1 (batched shallow ensemble, gmnn_api.cu): row tile rt = atom tile * heads + head holds dE^(head)/dG of the
    // atoms of tile rt / heads; Psi and sigma are the atom's, the adjoints go to row rt * 128 + tid of A.  N counts atoms
    // (rows of psi); dGt / A are then the batched buffers.
    const int64_t rtile = blockIdx.x * (int64_t)HALVES + hf;
    const int64_t tile = heads > 1 ? rtile / heads : rtile;
    const bool active = tile * TB < N;  // the last block of an odd tile count has an idle half
    const int64_t i = tile * TB + tid;
    const float *gt = dGt + rtile * (int64_t)(F::N * TB);  // this half's [F][128] tile

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
        float *dst = A + (rtile * TB + (ia - tile * TB)) * (int64_t)(NR * PSI);
        for (int q = lane; q < NR * PSI; q += 32) dst[q] = sP[q * CW + a];
    }
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
    const int heads = s->ens_batch > 1 ? s->ens_batch : 1;  // batched ensemble pass: dG / A of `heads` heads per atom tile
    const unsigned tiles = nblocks(s->n_rows, 128) * heads;
    k_contract_backward<NR, HALVES, LOCKSTEP, ORBIT><<<(tiles + HALVES - 1) / HALVES, 128 * HALVES, CbSmem<NR>::bytes(HALVES), st>>>(
        s->n_rows, s->psi, heads > 1 ? s->ens_dG : s->dG, s->pos4, s->model->scale, heads > 1 ? s->ens_A : s->A, s->row_atom,
        heads);
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
