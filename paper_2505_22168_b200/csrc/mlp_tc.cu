// mlp_tc.cu -- the per-atom MLP readout and its input gradient on the 5th-generation tensor cores
// (SURVEY.md 8(a) rows a7, a8; PAPER.md:63-65 Eq. 4, :153 forces by gradient).
//
//   mlp_precision = GMNN_MLP_3XTF32 : fp32-accurate.  a = a_hi + a_lo with a_hi = tf32(a) (round to
//       nearest), a_lo = a - a_hi (exact in fp32); a.b ~= a_lo.b_hi + a_hi.b_lo + a_hi.b_hi, three
//       kind::tf32 MMAs into one fp32 accumulator in tensor memory.  Dropped: a_lo.b_lo (<= 2^-22 |ab|)
//       and the bits of a_lo, b_lo below tf32 (<= 2^-22 |ab|): the same order as fp32 round-off.
//   mlp_precision = GMNN_MLP_TF32   : one kind::tf32 MMA per product.  Measured 1e-2 .. 2.5e-2 on the
//       force measure (rounding the operands to nearest instead of the tensor core's truncation does
//       not change that): not north_star's 2e-3 variant, kept as an unclaimed fast mode.
//
// The tensor core adds into its fp32 accumulator with truncation (measured: a 512-long chain of
// accumulating MMAs is biased towards zero by ~1e-5 relative), so the fp32-accurate mode keeps the
// chains short: the accumulator in tensor memory is flushed every `flush` pipeline stages into fp32
// REGISTER accumulators of the epilogue warps (round-to-nearest adds), and inside a stage the small
// cross terms are issued before the hi.hi terms so that they meet a small accumulator.
//
// One persistent, warp-specialised GEMM kernel  C[M][N] = A[M][K] . Bt[N][K]^T  with fused epilogues,
// on single CTAs (k_gemm_tc, 128 x bn tiles) or on CTA pairs (k_gemm_tc_pair, cta_group::2,
// 256 x bn tiles, each CTA holding half of the B rows):
//   warp 0        TMA producer into an NST-stage ring.  A: the tile-transposed activations
//                 ([M/128][K][128], every MLP matrix has this layout) as the MN-major operand, four
//                 {32 atoms, BK} boxes, 128-byte swizzle with 32-byte atoms (the only swizzle tcgen05
//                 accepts for an MN-major 32-bit operand).  B: weights, K-major; in 3xTF32 mode the hi
//                 and lo parts were split once at model creation (model->Ws / WTs, stacked [2N][K])
//                 and both are loaded
//   warp 1        allocates tensor memory; one lane issues tcgen05.mma (128 or 256 x bn x 8 each)
//   warps 4-7     (3xTF32) split the landed A tile: hi = tf32(a) in place, lo = a - hi beside it
//   warps 8-15    epilogue: drain each K chunk from tensor memory (two 256-column buffers in
//                 ping-pong, so draining chunk c overlaps the MMAs of chunk c+1) into 128 register
//                 accumulators per thread; after the last chunk bias + swish + swish' / gradient
//                 mask / head dot product, and coalesced stores into the tile-transposed output.
//                 setmaxnreg moves registers from the other warps to these.
// Activations stay fp32 in HBM, written once and read once (ncu: DRAM bytes = algorithmic bytes).
#include <cuda.h>
#include <cuda_fp16.h>

#include "gmnn_internal.h"
#include "tc_ptx.cuh"

namespace gmnn {

using namespace tc;

enum { EPI_PLAIN = 0, EPI_HIDDEN = 1, EPI_MUL = 2, EPI_HIDDEN_HEAD = 3 };
// Knock-out timing experiments (wrong results) exist only in builds with -DGMNN_EXPERIMENTS; the
// shipped library compiles them out.
#ifdef GMNN_EXPERIMENTS
#define TC_DBG(p) ((p).debug)
// cycle accounting of the CTA-pair kernel's roles (experiments build only): [EPI][CTA][slot]
__device__ long long g_tc_prof[4 * 160 * 8];
#define TC_PROF_DECL long long prof_[8] = {0, 0, 0, 0, 0, 0, 0, 0}
#define TC_PROF(slot, ...) { const long long t0_ = clock64(); __VA_ARGS__; prof_[slot] += clock64() - t0_; }
#define TC_PROF_BEGIN(name) const long long name = clock64()
#define TC_PROF_END(slot, name) prof_[slot] += clock64() - name
#define TC_PROF_FLUSH(epi) { for (int q_ = 0; q_ < 8; ++q_) if (prof_[q_]) atomicAdd((unsigned long long *)&g_tc_prof[((epi) * 160 + blockIdx.x) * 8 + q_], (unsigned long long)prof_[q_]); }
#else
#define TC_DBG(p) 0
#define TC_PROF_DECL
#define TC_PROF(slot, ...) { __VA_ARGS__; }
#define TC_PROF_BEGIN(name)
#define TC_PROF_END(slot, name)
#define TC_PROF_FLUSH(epi)
#endif
// EPI_HIDDEN_HEAD: last hidden layer of a single-head model.  h = swish(z) is not stored (the backward
// needs only swish'); its dot product with the head weights is: every thread writes the partial sum
// over its columns to ypart[slot][atom], slot = 2 * column tile + column half, and k_heads_finish
// adds the slots in order.

constexpr int TC_BM = 128;           // rows of A per tile = TMEM lanes
constexpr int TC_BN_MAX = 256;       // columns per accumulator buffer
constexpr int TC_THREADS = 16 * 32;  // four warpgroups: control, splitters, 2 x epilogue
constexpr int TC_FIRST_SPLIT_WARP = 4;
constexpr int TC_FIRST_EPI_WARP = 8;
constexpr int TC_REGS_CONTROL = 40, TC_REGS_SPLIT = 64, TC_REGS_EPI = 200;  // 128 * (40 + 64 + 2 * 200) <= 65536
constexpr int TC_STAGE_BYTES_TOTAL = 192 * 1024;
#ifndef TC_EB
#define TC_EB 16  // columns per batch of the fused epilogue
#endif

template <bool SPLIT, int BK>
struct TcCfg {
    static constexpr int SWZ = BK * 4;                           // bytes per tile row = swizzle span
    static constexpr int A_BYTES = TC_BM * BK * 4;
    static constexpr int B_BYTES = TC_BN_MAX * BK * 4;
    static constexpr int STAGE_BYTES = (A_BYTES + B_BYTES) * (SPLIT ? 2 : 1);
    static constexpr int NST = TC_STAGE_BYTES_TOTAL / STAGE_BYTES;
    static constexpr int SMEM_BYTES = NST * STAGE_BYTES + 1024 /*alignment slack*/ + 512 /*barriers*/;
    static_assert(NST >= 2, "pipeline needs at least two stages");
};

struct TcArgs {
    int M, N, K;
    int bn;        // columns per tile (multiple of 16, <= 256)
    int n_tiles_n;
    int n_tiles;   // total
    int flush;     // pipeline stages per accumulator flush (K chunk = flush * BK)
    int flush1;    // ... of the first two chunks of a tile (>= flush)
    int xy;        // CTA-pair kernels: 0 = ping-pong of mixed chunks (backward GEMMs), 1 = cross terms and hi.hi terms in accumulators
                   // of their own, 2 = ping-pong of chunks whose cross terms all precede their hi.hi terms (forward GEMMs)
    int order;     // CTA-pair kernels: 0 = tiles dealt round-robin to the pairs, 1 = a pair runs the column tiles of a row tile back to back
    int dmul_pf;   // EPI_MUL: the multiplier block of a tile is prefetched into L2 this many pipeline stages before the tile's last (< 0: never)
    int debug;     // -DGMNN_EXPERIMENTS builds only (results wrong): 1 skip split work, 2 hi.hi MMA only, 4 skip the elementwise
                   // and the stores, 8 skip the stores only, 16 skip the tensor-memory drains
    float *C;      // [M][N]
    float *C2;     // EPI_HIDDEN: swish'(z)
    const float *bias;
    const float *Dmul;  // EPI_MUL: [M][N]; batched ensemble backward: row tile rt reads row tile rt / dmul_row_div and column
                        // c reads column c % dmul_N of a multiplier that is [M / dmul_row_div][dmul_N]
    int dmul_N, dmul_row_div;
    const float *w_head;  // EPI_HIDDEN_HEAD: [N] weights of the single head
    float *ypart;         // EPI_HIDDEN_HEAD: [2 * n_tiles_n][m_pad]
    int64_t m_pad;
    // 3xFP16: absolute maxima (fp32 bit patterns, device scalars) of A and of the fp32 matrix behind Bt;
    // amax_out (may be null) receives the maximum of what this GEMM stores in C
    const uint32_t *amax_a, *amax_b;
    uint32_t *amax_out;
};

// Accumulator-flush schedule of a tile: the first two chunks span flush1 pipeline stages each, the
// rest `flush`.  (Longer first chunks give the MMA issuer more run-way while the epilogue warps are
// still in the previous tile's final phase; used by the backward GEMMs, see tc_gemm.)
__device__ __forceinline__ void chunk_pos(const TcArgs &p, int kb, int nkb, bool &first, bool &last) {
    const int head = 2 * p.flush1;
    const int pos = kb < head ? kb % p.flush1 : (kb - head) % p.flush;
    const int len = kb < head ? p.flush1 : p.flush;
    first = pos == 0;
    last = pos == len - 1 || kb == nkb - 1;
}
__device__ __forceinline__ int chunk_count(const TcArgs &p, int nkb) {
    const int head = nkb < 2 * p.flush1 ? nkb : 2 * p.flush1;
    return (head + p.flush1 - 1) / p.flush1 + (nkb - head + p.flush - 1) / p.flush;
}

__device__ __forceinline__ void swish_pair_tc(float z, float &h, float &d) {
    const float s = __fdividef(1.f, 1.f + __expf(-z));  // ex2.approx + rcp.approx: ~2 ulp, no slow path
    h = z * s;
    d = s * (1.f + z * (1.f - s));
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// swish and swish' of z = a * zs from the raw accumulator a (which already carries the bias, see tc_init_acc):
// t = a * (-zs log2 e) -> e^-z = ex2(t); s = 1 / (1 + e^-z); h = z s; d = s + h (1 - s) = fma(-h, s, s + h).
// Eight issue slots and two MUFU per element (the final phase of a forward tile is bound by exactly these).
__device__ __forceinline__ void swish_pair_acc(float a, float zs, float k1, float &h, float &d) {
    const float z = a * zs;
    const float s = rcp_approx(1.f + ex2_approx(a * k1));
    h = z * s;
    d = fmaf(-h, s, s + h);
}

// hi = tf32(x) (round to nearest) in place, lo = x - hi beside it, for `n4` float4 of one operand
// tile, by 128 threads.  Eight independent loads are issued before the first store: hi and lo tiles
// may alias as far as the compiler knows, so a plain loop would serialise load -> store -> load.
__device__ __forceinline__ void split_hi_lo(float4 *hi, float4 *lo, int n4, int tid) {
    for (int q0 = tid; q0 < n4; q0 += 8 * 128) {
        float4 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (q0 + u * 128 < n4) v[u] = hi[q0 + u * 128];
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (q0 + u * 128 < n4) {
                float4 h, l;
                h.x = to_tf32_rna(v[u].x); h.y = to_tf32_rna(v[u].y); h.z = to_tf32_rna(v[u].z); h.w = to_tf32_rna(v[u].w);
                l.x = v[u].x - h.x; l.y = v[u].y - h.y; l.z = v[u].z - h.z; l.w = v[u].w - h.w;
                hi[q0 + u * 128] = h;
                lo[q0 + u * 128] = l;
            }
    }
}

// Fused elementwise and stores of one finished tile held in the epilogue warps' registers.
// SCALED (3xFP16): the accumulator is multiplied by `oscale` first, and `tmax` follows the largest
// magnitude stored in C (the next GEMM's operand scale).
template <int EPI, bool SCALED = false>
__device__ __forceinline__ void tc_store_tile(const TcArgs &p, float (&acc)[4][32], int m0, int n0, int quad, int lane,
                                              int half, int n_groups, bool row_ok, float oscale, float &tmax) {
    // every matrix the MLP touches is tile-transposed, [M / 128][N][128]: column c of this tile is
    // 128 consecutive floats, so each warp store / load below is one full 128-byte line.  The stores are streaming
    // (st.global.cs): the outputs are 1.5 - 4 GB that only the next kernel reads, and left to the default policy
    // their dirty lines push the activation boxes out of L2 between the reads of the two column tiles of a row tile
    const int64_t tbase = (int64_t)(m0 / TC_BM) * p.N * TC_BM + quad * 32 + lane;
    float *__restrict__ Cout = p.C;
    float *__restrict__ C2out = p.C2;
    const float *__restrict__ bias = p.bias;
    const float *__restrict__ Dmul = p.Dmul;
    float ysum = 0.f;
#pragma unroll
    for (int gi = 0; gi < 4; ++gi) {
        const int g = 2 * gi + half;
        const int col0 = n0 + g * 32;
        if (g >= n_groups || !row_ok || (TC_DBG(p) & 4)) continue;
        // TC_EB columns at a time: loads first, then the arithmetic, then the stores, so that the
        // dependency chains (ex2, rcp, fma; DRAM latency of the multiplier) overlap
#pragma unroll
        for (int j0 = 0; j0 < 32; j0 += TC_EB) {
            if (col0 + j0 >= p.N || g * 32 + j0 >= p.bn) continue;
            // N and bn are multiples of 8: the second half of a 16-wide batch may be absent
            const int nc = (col0 + j0 + TC_EB <= p.N && g * 32 + j0 + TC_EB <= p.bn) ? TC_EB : 8;
            const int64_t o = tbase + (int64_t)(col0 + j0) * TC_BM;
            float in[TC_EB], h[TC_EB], d[TC_EB];
            if (EPI == EPI_HIDDEN_HEAD) {
                float wh[TC_EB];
#pragma unroll
                for (int c = 0; c < TC_EB; ++c) {
                    in[c] = c < nc ? __ldg(bias + col0 + j0 + c) : 0.f;
                    wh[c] = c < nc ? __ldg(p.w_head + col0 + j0 + c) : 0.f;
                }
#pragma unroll
                for (int c = 0; c < TC_EB; ++c) swish_pair_tc(SCALED ? fmaf(acc[gi][j0 + c], oscale, in[c]) : acc[gi][j0 + c] + in[c], h[c], d[c]);
#pragma unroll
                for (int c = 0; c < TC_EB; ++c)
                    if (c < nc) {
                        ysum = fmaf(h[c], wh[c], ysum);
                        if (TC_DBG(p) & 8) {
                            tmax = fmaxf(tmax, d[c]);
                            continue;
                        }
                        __stcs(C2out + o + c * TC_BM, d[c]);
                    }
            } else if (EPI == EPI_HIDDEN) {
#pragma unroll
                for (int c = 0; c < TC_EB; ++c) in[c] = c < nc ? __ldg(bias + col0 + j0 + c) : 0.f;
#pragma unroll
                for (int c = 0; c < TC_EB; ++c) swish_pair_tc(SCALED ? fmaf(acc[gi][j0 + c], oscale, in[c]) : acc[gi][j0 + c] + in[c], h[c], d[c]);
#pragma unroll
                for (int c = 0; c < TC_EB; ++c)
                    if (c < nc) {
                        if (TC_DBG(p) & 8) {  // knock-out: arithmetic without the stores
                            tmax = fmaxf(tmax, fabsf(h[c]) + d[c]);
                            continue;
                        }
                        __stcs(Cout + o + c * TC_BM, h[c]);
                        __stcs(C2out + o + c * TC_BM, d[c]);
                        if (SCALED) tmax = fmaxf(tmax, fabsf(h[c]));
                    }
            } else if (EPI == EPI_MUL) {
                const int64_t om = (int64_t)((m0 / TC_BM) / p.dmul_row_div) * p.dmul_N * TC_BM + quad * 32 + lane +
                                   (int64_t)((col0 + j0) % p.dmul_N) * TC_BM;
#pragma unroll
                for (int c = 0; c < TC_EB; ++c) in[c] = c < nc ? __ldg(Dmul + om + c * TC_BM) : 0.f;
#pragma unroll
                for (int c = 0; c < TC_EB; ++c)
                    if (c < nc) {
                        const float v = (SCALED ? acc[gi][j0 + c] * oscale : acc[gi][j0 + c]) * in[c];
                        if (SCALED) tmax = fmaxf(tmax, fabsf(v));
                        if (TC_DBG(p) & 8) continue;
                        __stcs(Cout + o + c * TC_BM, v);
                    }
            } else {
#pragma unroll
                for (int c = 0; c < TC_EB; ++c)
                    if (c < nc) __stcs(Cout + o + c * TC_BM, SCALED ? acc[gi][j0 + c] * oscale : acc[gi][j0 + c]);
            }
        }
    }
    if (EPI == EPI_HIDDEN_HEAD && row_ok && !(TC_DBG(p) & 4))
        p.ypart[(int64_t)(2 * (n0 / p.bn) + half) * p.m_pad + m0 + quad * 32 + lane] = ysum;
}


// ---- epilogue of the CTA-pair kernels ------------------------------------------------------------------------------
// The forward bias is folded into the register accumulators when a tile starts (acc = bias / oscale, while the first MMAs
// of the tile run), so the final phase has no loads; every thread keeps base pointers of its row, so the stores take
// immediate column offsets.  Valid columns of a 32-column group: multiples of 8 (N and bn are).
__device__ __forceinline__ int tc_group_valid(const TcArgs &p, int n0, int g) {
    int v = p.N - (n0 + g * 32);
    const int w = p.bn - g * 32;
    v = v < w ? v : w;
    return v < 0 ? 0 : (v > 32 ? 32 : v);
}

template <int EPI>
__device__ __forceinline__ void tc_init_acc(const TcArgs &p, float (&acc)[4][32], int n0, int half, float inv_oscale) {
#pragma unroll
    for (int gi = 0; gi < 4; ++gi) {
        const int g = 2 * gi + half;
        const int nv = (EPI == EPI_HIDDEN || EPI == EPI_HIDDEN_HEAD) ? tc_group_valid(p, n0, g) : 0;
        const float4 *__restrict__ b = reinterpret_cast<const float4 *>(p.bias + n0 + g * 32);  // 16-byte aligned: n0, widths % 16 == 0
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const float4 t = 4 * q < nv ? __ldg(b + q) : make_float4(0.f, 0.f, 0.f, 0.f);
            acc[gi][4 * q] = t.x * inv_oscale, acc[gi][4 * q + 1] = t.y * inv_oscale;
            acc[gi][4 * q + 2] = t.z * inv_oscale, acc[gi][4 * q + 3] = t.w * inv_oscale;
        }
    }
}

template <int EPI, bool SCALED>
__device__ __forceinline__ void tc_finish_tile(const TcArgs &p, float (&acc)[4][32], int m0, int n0, int quad, int lane,
                                               int half, bool row_ok, float oscale, float &tmax) {
    // forward epilogues (EPI_HIDDEN, EPI_HIDDEN_HEAD).  Tile-transposed [M / 128][N][128]: column c of this tile is 128
    // consecutive floats, each warp store one full 128-byte line at a compile-time offset from the thread's base pointer.
    const int64_t tbase = (int64_t)(m0 / TC_BM) * p.N * TC_BM + quad * 32 + lane + (int64_t)(n0 + half * 32) * TC_BM;
    float *__restrict__ cp = p.C + tbase;
    float *__restrict__ dp = p.C2 + tbase;
    const float k1 = -oscale * 1.4426950408889634f;
    float ysum = 0.f;
    if (row_ok && !(TC_DBG(p) & 4)) {
#pragma unroll
        for (int gi = 0; gi < 4; ++gi) {
            const int g = 2 * gi + half;
            const int nv = tc_group_valid(p, n0, g);
            const float *__restrict__ wh = p.w_head + n0 + g * 32;
#pragma unroll
            for (int j0 = 0; j0 < 32; j0 += 8) {
                if (j0 >= nv) continue;  // warp-uniform
                float h[8], d[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) swish_pair_acc(acc[gi][j0 + c], oscale, k1, h[c], d[c]);
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const int off = (gi * 64 + j0 + c) * TC_BM;  // compile-time column offset of the store
                    if (EPI == EPI_HIDDEN_HEAD) ysum = fmaf(h[c], __ldg(wh + j0 + c), ysum);
                    if (SCALED && EPI == EPI_HIDDEN) tmax = fmaxf(tmax, fabsf(h[c]));
                    if (TC_DBG(p) & 8) {  // knock-out: arithmetic without the stores
                        tmax = fmaxf(tmax, d[c]);
                        continue;
                    }
                    if (EPI == EPI_HIDDEN) __stcs(cp + off, h[c]);
                    __stcs(dp + off, d[c]);
                }
            }
        }
        if (EPI == EPI_HIDDEN_HEAD) p.ypart[(int64_t)(2 * (n0 / p.bn) + half) * p.m_pad + m0 + quad * 32 + lane] = ysum;
    }
}

template <bool SPLIT, int BK, int EPI>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_gemm_tc(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const TcArgs p) {
    using Cfg = TcCfg<SPLIT, BK>;
    constexpr int NST = Cfg::NST;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    // stage s: [A_hi | A_lo (SPLIT) | B_hi | B_lo (SPLIT)]
    auto a_hi = [&](int s) { return smem_base + (uint32_t)s * Cfg::STAGE_BYTES; };
    auto a_lo = [&](int s) { return a_hi(s) + Cfg::A_BYTES; };
    auto b_hi = [&](int s) { return a_hi(s) + Cfg::A_BYTES * (SPLIT ? 2 : 1); };
    auto b_lo = [&](int s) { return b_hi(s) + Cfg::B_BYTES; };
    const uint32_t bar_base = smem_base + (uint32_t)NST * Cfg::STAGE_BYTES;
    auto bar_full = [&](int s) { return bar_base + 8u * s; };
    auto bar_split = [&](int s) { return bar_base + 8u * (NST + s); };
    auto bar_empty = [&](int s) { return bar_base + 8u * (2 * NST + s); };
    auto bar_tfull = [&](int a) { return bar_base + 8u * (3 * NST + a); };
    auto bar_tempty = [&](int a) { return bar_base + 8u * (3 * NST + 2 + a); };
    const uint32_t tmem_slot = bar_base + 8u * (3 * NST + 4);
    volatile uint32_t *tmem_slot_gen = reinterpret_cast<volatile uint32_t *>(smem_gen + (size_t)NST * Cfg::STAGE_BYTES + 8 * (3 * NST + 4));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nkb = (p.K + BK - 1) / BK;  // pipeline stages per tile; chunk c covers stages [c*flush, (c+1)*flush)

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmB);
        for (int s = 0; s < NST; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_split(s), 4);
            mbar_init(bar_empty(s), 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull(a), 1);
            mbar_init(bar_tempty(a), 8);
        }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc<512>(tmem_slot);
    tcgen05_fence_before();
    __syncthreads();
    tcgen05_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;

    if (warp < TC_FIRST_SPLIT_WARP) {
        setmaxnreg_dec<TC_REGS_CONTROL>();
        if (warp == 0 && lane == 0) {
            // ===== TMA producer =====
            const uint32_t tx = (uint32_t)(Cfg::A_BYTES + p.bn * BK * 4 * (SPLIT ? 2 : 1));
            uint32_t it = 0;
            for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
                const int m0 = (t / p.n_tiles_n) * TC_BM, n0 = (t % p.n_tiles_n) * p.bn;
                for (int kb = 0; kb < nkb; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(bar_empty(s), ((it / NST) & 1) ^ 1);
                    mbar_arrive_expect_tx(bar_full(s), tx);
                    for (int q = 0; q < 4; ++q)  // four 32-atom column blocks of the tile, [BK][32 floats] each
                        tma_load_2d(a_hi(s) + q * (BK * 128), &tmA, bar_full(s), q * 32, (m0 / TC_BM) * p.K + kb * BK);
                    tma_load_2d(b_hi(s), &tmB, bar_full(s), kb * BK, n0);
                    if (SPLIT) tma_load_2d(b_lo(s), &tmB, bar_full(s), kb * BK, p.N + n0);  // lo rows follow the N hi rows
                }
            }
        } else if (warp == 1 && lane == 0) {
            // ===== MMA issuer =====
            const uint32_t idesc = make_idesc_tf32(TC_BM, p.bn, true);
            uint32_t it = 0, chunk = 0;
            for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
                for (int kb = 0; kb < nkb; ++kb, ++it) {
                    bool chunk_first, chunk_last;
                    chunk_pos(p, kb, nkb, chunk_first, chunk_last);
                    const int a = chunk & 1;
                    const uint32_t d_tmem = tmem_base + (uint32_t)a * TC_BN_MAX;
                    if (chunk_first) {
                        mbar_wait(bar_tempty(a), ((chunk >> 1) & 1) ^ 1);
                        tcgen05_fence_after();
                    }
                    const int s = it % NST;
                    mbar_wait(SPLIT ? bar_split(s) : bar_full(s), (it / NST) & 1);
                    tcgen05_fence_after();
                    const int krem = p.K - kb * BK;
                    const int ksteps = krem >= BK ? BK / 8 : (krem + 7) / 8;
                    const uint64_t da_hi = make_smem_desc_mn128(a_hi(s), BK * 128), db_hi = make_smem_desc<Cfg::SWZ>(b_hi(s));
                    uint32_t acc = !chunk_first;
                    if (SPLIT && !(TC_DBG(p) & 2)) {  // small cross terms first: they meet the smallest accumulator
                        const uint64_t da_lo = make_smem_desc_mn128(a_lo(s), BK * 128), db_lo = make_smem_desc<Cfg::SWZ>(b_lo(s));
                        for (int k = 0; k < ksteps; ++k) {
                            const uint64_t koff = (uint64_t)((k * 32) >> 4);    // B: 8 tf32 = 32 bytes along the row
                            const uint64_t aoff = (uint64_t)((k * 1024) >> 4);  // A: 8 k rows = one 1024-byte atom
                            mma_tf32_ss(d_tmem, da_lo + aoff, db_hi + koff, idesc, acc);
                            mma_tf32_ss(d_tmem, da_hi + aoff, db_lo + koff, idesc, 1u);
                            acc = 1u;
                        }
                    }
                    for (int k = 0; k < ksteps; ++k) {
                        const uint64_t koff = (uint64_t)((k * 32) >> 4), aoff = (uint64_t)((k * 1024) >> 4);
                        mma_tf32_ss(d_tmem, da_hi + aoff, db_hi + koff, idesc, acc);
                        acc = 1u;
                    }
                    mma_commit(bar_empty(s));
                    if (chunk_last) {
                        mma_commit(bar_tfull(a));
                        ++chunk;
                    }
                }
            }
        }
    } else if (warp < TC_FIRST_EPI_WARP) {
        setmaxnreg_dec<TC_REGS_SPLIT>();
        // ===== splitters (3xTF32): hi = tf32(x) in place, lo = x - hi beside it =====
        if (SPLIT) {
            const int tid = threadIdx.x - TC_FIRST_SPLIT_WARP * 32;  // 0..127
            const int n_a4 = Cfg::A_BYTES / 16;
            uint32_t it = 0;
            for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
                for (int kb = 0; kb < nkb; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(bar_full(s), (it / NST) & 1);
                    float4 *ah = reinterpret_cast<float4 *>(smem_gen + (size_t)s * Cfg::STAGE_BYTES);
                    float4 *al = reinterpret_cast<float4 *>(smem_gen + (size_t)s * Cfg::STAGE_BYTES + Cfg::A_BYTES);
                    if (!(TC_DBG(p) & 1)) split_hi_lo(ah, al, n_a4, tid);  // B arrives split (model->Ws / WTs)
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_split(s));
                }
            }
        }
    } else {
        setmaxnreg_inc<TC_REGS_EPI>();
        // ===== epilogue: drain K chunks TMEM -> register accumulators, then the fused elementwise =====
        const int quad = warp & 3;                        // TMEM lanes 32*quad .. 32*quad+31
        const int half = (warp - TC_FIRST_EPI_WARP) >> 2;  // 32-column groups half, half+2, half+4, half+6
        const int n_groups = (p.bn + 31) / 32;
        const int n_chunks = chunk_count(p, nkb);
        const uint32_t lane_base = tmem_base + ((uint32_t)(quad * 32) << 16);
        uint32_t chunk = 0;
        for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
            const int m0 = (t / p.n_tiles_n) * TC_BM, n0 = (t % p.n_tiles_n) * p.bn;
            const int row = m0 + quad * 32 + lane;
            const bool row_ok = row < p.M;
            float acc[4][32];
#pragma unroll
            for (int gi = 0; gi < 4; ++gi)
#pragma unroll
                for (int j = 0; j < 32; ++j) acc[gi][j] = 0.f;
            for (int c = 0; c < n_chunks; ++c, ++chunk) {
                const int a = chunk & 1;
                mbar_wait(bar_tfull(a), (chunk >> 1) & 1);
                tcgen05_fence_after();
#pragma unroll
                for (int gi = 0; gi < 4; ++gi) {
                    const int g = 2 * gi + half;
                    if (g < n_groups) {
                        uint32_t v[32];
                        tmem_ld_32x32(lane_base + (uint32_t)(a * TC_BN_MAX + g * 32), v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 32; ++j) acc[gi][j] += __uint_as_float(v[j]);
                    }
                }
                tcgen05_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_tempty(a));
            }
            float unused = 0.f;
            tc_store_tile<EPI>(p, acc, m0, n0, quad, lane, half, n_groups, row_ok, 1.f, unused);
        }
    }

    tcgen05_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem_base);
}

static int tc_num_sms();

// ---- CTA-pair variant of the 3xTF32 kernel (cta_group::2) ------------------------------------------
// Two CTAs of a cluster (one per SM of a TPC) work on a 256 x bn tile: each holds its own 128 rows of A
// and HALF of the bn rows of B in shared memory, splits them into hi / lo itself, and owns the 128 x bn
// accumulator rows in its tensor memory.  One thread of the leader CTA (cluster rank 0) issues the
// M = 256 MMAs for both.  Per SM this halves the B bytes loaded from L2, split by the splitter warps and
// read by the tensor core, which is what bounds the single-CTA kernel (shared-memory bandwidth).
// Hand-shakes across the pair: split-done and accumulator-drained arrivals go to the leader's
// barriers (mapa + remote arrive); the leader's tcgen05.commit multicasts to both CTAs' barriers.
// Accumulators.  The tensor core adds into its fp32 accumulator with truncation, so long accumulation chains of LARGE
// terms bias the result.  The three products of the split are therefore kept apart: the cross terms
// a_lo.b_hi + a_hi.b_lo, 2^-11 of the result, go to accumulator X (tensor-memory columns [0, 256)) for the whole K range of a
// tile -- their truncation errors are 2^-11 of the hi.hi ones -- and only the hi.hi terms go to accumulator Y (columns
// [256, 512)), which the epilogue warps drain into fp32 registers (round-to-nearest adds) every p.flush pipeline stages.  Y is
// single-buffered: while it is drained the MMA pipe runs the next stage's cross terms, and during the final phase of a
// tile (elementwise + stores) the issuer has a whole group of stages plus one stage of cross terms of run-way.
// F16 = true is the 3xFP16 mode (GMNN_MLP_3XF16): the same three-product split on kind::f16, whose
// MMAs run at twice the tf32 rate on half the operand bytes.  a' = a * 2^s with 2^14 <= max |a'| < 2^15
// (s from the matrix's absolute maximum, a device scalar the producing kernel left), hi = fp16(a'),
// lo = fp16(a' - hi): 22 significand bits like the tf32 split; elements below 2^-18 of the maximum lose
// relative (not absolute: <= 2^-40 of the maximum) accuracy to the fp16 exponent range.  The splitter
// warps read the fp32 A tile where TMA landed it ([BK][128 atoms], not swizzled) and write hi / lo as
// K-major fp16 rows in the 128- or 64-byte swizzle; B arrives split and scaled (model->Wh / WTh).  The
// epilogue multiplies the accumulator by 2^-(s_a + s_b).
template <bool F16, int BK>
struct TcPairCfg {
    static constexpr int ES = F16 ? 2 : 4;                          // operand element size
    static constexpr int ROWB = BK * ES;                            // bytes per K-major operand row = swizzle span
    static constexpr int LAND_BYTES = 0;                            // (F16: the fp32 A tile lands where hi and lo will be)
    static constexpr int A_BYTES = TC_BM * BK * ES;
    static constexpr int B_BYTES = (TC_BN_MAX / 2) * BK * ES;       // this CTA's half of the B tile
    static constexpr int STAGE_BYTES = LAND_BYTES + 2 * (A_BYTES + B_BYTES);  // hi and lo of both
    static constexpr int NST = TC_STAGE_BYTES_TOTAL / STAGE_BYTES;
    static constexpr int SMEM_BYTES = NST * STAGE_BYTES + 1024 + 512;
    static constexpr int KSTEP = 32 / ES;                           // K per MMA instruction
    // registers per thread of the control / splitter / epilogue warpgroups (setmaxnreg; 128 x sum <= 65536)
    static constexpr int REGS_CONTROL = F16 ? 32 : TC_REGS_CONTROL, REGS_SPLIT = F16 ? 96 : TC_REGS_SPLIT,
                         REGS_EPI = F16 ? 192 : TC_REGS_EPI;
    static_assert(NST >= 2, "pipeline needs at least two stages");
};

// 2^e for the fp16 split: e = 14 - floor(log2(amax)), clamped so that all scales stay normal numbers
__device__ __forceinline__ int amax_exponent(uint32_t bits) {
    int e = bits ? (int)(bits >> 23) - 127 : 0;
    return e < -40 ? -40 : (e > 40 ? 40 : e);
}
__device__ __forceinline__ float pow2i(int e) { return __int_as_float((127 + e) << 23); }

// fp32 A tile [BK][128] -> hi / lo fp16 rows (K-major, swizzled) IN PLACE, one atom (row) per thread of the
// four splitter warps: every thread reads its column (conflict-free: lanes are consecutive atoms) and
// converts it in registers; after a barrier among the 128 threads the rows are written over the tile
// (hi rows in the first half, lo rows in the second).
template <int BK>
__device__ __forceinline__ void split_f16_tile(uint8_t *__restrict__ stage, int m, float scale, int k_valid) {
    constexpr int ROWB = BK * 2;
    const float *land = reinterpret_cast<const float *>(stage);
    uint32_t h[BK / 2], l[BK / 2];
#pragma unroll
    for (int q = 0; q < BK / 2; ++q) {
        const bool ok = (2 * q) < k_valid;  // K is a multiple of 8: an 8-wide chunk is whole or absent
        const float a = ok ? land[(2 * q) * TC_BM + m] * scale : 0.f, b = ok ? land[(2 * q + 1) * TC_BM + m] * scale : 0.f;
        const __half2 hh = __floats2half2_rn(a, b);
        const float2 hf = __half22float2(hh);
        const __half2 ll = __floats2half2_rn(a - hf.x, b - hf.y);
        h[q] = *reinterpret_cast<const uint32_t *>(&hh);
        l[q] = *reinterpret_cast<const uint32_t *>(&ll);
    }
    asm volatile("bar.sync 1, 128;" ::: "memory");  // all columns read before any row is written
#pragma unroll
    for (int c = 0; c < BK / 8; ++c) {
        uint32_t o = (uint32_t)(m * ROWB + c * 16);
        o ^= ((o >> 7) & (uint32_t)(ROWB / 16 - 1)) << 4;  // 128- / 64-byte swizzle of the 16-byte chunk index
        *reinterpret_cast<uint4 *>(stage + o) = make_uint4(h[4 * c], h[4 * c + 1], h[4 * c + 2], h[4 * c + 3]);
        *reinterpret_cast<uint4 *>(stage + TC_BM * ROWB + o) = make_uint4(l[4 * c], l[4 * c + 1], l[4 * c + 2], l[4 * c + 3]);
    }
}

template <bool F16, int BK, int EPI>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(TC_THREADS, 1)
k_gemm_tc_pair(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const TcArgs p) {
    using Cfg = TcPairCfg<F16, BK>;
    constexpr int NST = Cfg::NST;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;  // identical offset in both CTAs
    uint8_t *smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    // stage: [A_hi | A_lo | B_hi | B_lo]; the fp32 A tile of the 3xFP16 mode lands on A_hi | A_lo
    auto a_hi = [&](int s) { return smem_base + (uint32_t)s * Cfg::STAGE_BYTES + Cfg::LAND_BYTES; };
    auto a_lo = [&](int s) { return a_hi(s) + Cfg::A_BYTES; };
    auto b_hi = [&](int s) { return a_hi(s) + 2 * Cfg::A_BYTES; };
    auto b_lo = [&](int s) { return b_hi(s) + Cfg::B_BYTES; };
    const uint32_t bar_base = smem_base + (uint32_t)NST * Cfg::STAGE_BYTES;
    auto bar_full = [&](int s) { return bar_base + 8u * s; };               // own TMA landed
    auto bar_split = [&](int s) { return bar_base + 8u * (NST + s); };      // leader's: both CTAs split
    auto bar_empty = [&](int s) { return bar_base + 8u * (2 * NST + s); };  // own: MMAs of the stage done
    auto bar_tfull = [&](int a) { return bar_base + 8u * (3 * NST + a); };  // own: chunk complete
    auto bar_tempty = [&](int a) { return bar_base + 8u * (3 * NST + 2 + a); };  // leader's: both drained
    const uint32_t tmem_slot = bar_base + 8u * (3 * NST + 4);
    volatile uint32_t *tmem_slot_gen = reinterpret_cast<volatile uint32_t *>(smem_gen + (size_t)NST * Cfg::STAGE_BYTES + 8 * (3 * NST + 4));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const int nkb = (p.K + BK - 1) / BK;
    const int hb = p.bn >> 1;  // B rows held by each CTA

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmA);
        tma_prefetch_desc(&tmB);
        for (int s = 0; s < NST; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_split(s), 8);   // 4 splitter warps x 2 CTAs
            mbar_init(bar_empty(s), 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull(a), 1);
            mbar_init(bar_tempty(a), 16);  // 8 epilogue warps x 2 CTAs
        }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc_pair<512>(tmem_slot);
    tcgen05_fence_before();
    cluster_sync_all();  // barriers of both CTAs initialised before any remote arrive
    tcgen05_fence_after();
    const uint32_t tmem_base = *tmem_slot_gen;

    // Tile order.  p.order = 0: tile t of the launch goes to pair t % n_pairs, so that the column tiles of one row tile run
    // on neighbouring pairs at about the same time.  p.order = 1: a pair takes whole row tiles and runs their column tiles
    // back to back, so that the second read of the row tile's activation boxes follows the first by one tile time whatever
    // the drift between pairs.
    const int n_row_tiles = p.n_tiles / p.n_tiles_n;
    const int t_end = p.order ? ((n_row_tiles + n_pairs - 1) / n_pairs) * p.n_tiles_n * n_pairs : p.n_tiles;
    auto tile_of = [&](int tt) {
        if (!p.order) return tt;
        const int k = tt / n_pairs;
        return ((k / p.n_tiles_n) * n_pairs + pair) * p.n_tiles_n + k % p.n_tiles_n;
    };

    if (warp < TC_FIRST_SPLIT_WARP) {
        setmaxnreg_dec<Cfg::REGS_CONTROL>();
        if (warp == 0 && lane == 0) {
            // ===== TMA producer: own A rows, own half of B =====
            const uint32_t tx = (uint32_t)(TC_BM * BK * 4 + 2 * hb * BK * Cfg::ES);
            TC_PROF_DECL;
            uint32_t it = 0;
            const int pf_kb = p.dmul_pf < 0 ? -1 : (nkb - 1 - p.dmul_pf > 0 ? nkb - 1 - p.dmul_pf : 0);
            TC_PROF_BEGIN(t_all);
            for (int tt = pair; tt < t_end; tt += n_pairs) {
                const int t = tile_of(tt);
                if (t >= p.n_tiles) continue;  // same decision in every role of both CTAs
                const int mt = 2 * (t / p.n_tiles_n) + (int)rank, n0 = (t % p.n_tiles_n) * p.bn;
                for (int kb = 0; kb < nkb; ++kb, ++it) {
                    const int s = it % NST;
                    if (EPI == EPI_MUL && kb == pf_kb && (int64_t)mt * TC_BM < p.M) {
                        // the multiplier block of this tile (swish' of the layer below: bn columns x 128 rows, contiguous) is read
                        // by the epilogue at the END of the tile, from HBM: bring it into L2 shortly before that (measured at
                        // config 5: issued at the start of the tile the block is evicted again before its use, 7.4 GB of DRAM
                        // reads per launch instead of 5.3; at the last stage 5.4 GB and 3 % less time than without)
                        const int cols = p.N - n0 < p.bn ? p.N - n0 : p.bn;
                        const char *blk = reinterpret_cast<const char *>(
                            p.Dmul + ((int64_t)(mt / p.dmul_row_div) * p.dmul_N + n0 % p.dmul_N) * TC_BM);
                        for (int c = 0; c < cols; c += 64) bulk_prefetch_l2(blk + (int64_t)c * TC_BM * 4, (uint32_t)((cols - c < 64 ? cols - c : 64) * TC_BM * 4));
                    }
                    TC_PROF(0, mbar_wait(bar_empty(s), ((it / NST) & 1) ^ 1));
                    mbar_arrive_expect_tx(bar_full(s), tx);
                    if (F16) {
                        tma_load_2d(a_hi(s), &tmA, bar_full(s), 0, mt * p.K + kb * BK);  // [BK][128] fp32
                    } else {
                        for (int q = 0; q < 4; ++q)
                            tma_load_2d(a_hi(s) + q * (BK * 128), &tmA, bar_full(s), q * 32, mt * p.K + kb * BK);
                    }
                    tma_load_2d(b_hi(s), &tmB, bar_full(s), kb * BK, n0 + (int)rank * hb);
                    tma_load_2d(b_lo(s), &tmB, bar_full(s), kb * BK, p.N + n0 + (int)rank * hb);  // lo rows follow the hi rows
                }
            }
            TC_PROF_END(5, t_all);
            TC_PROF_FLUSH(EPI);
        } else if (warp == 1 && lane == 0 && rank == 0) {
            // ===== MMA issuer (leader CTA only) =====
            // Two accumulators in tensor memory (see the header of this kernel): X, columns [0, 256), takes the cross terms
            // a_lo.b_hi + a_hi.b_lo of the WHOLE K range of a tile and is drained once per tile; Y, columns [256, 512), takes the
            // hi.hi terms and is drained every p.flush pipeline stages.
            const uint32_t idesc = F16 ? make_idesc_f16(2 * TC_BM, p.bn) : make_idesc_tf32(2 * TC_BM, p.bn, true);
            const uint32_t d_x = tmem_base, d_y = tmem_base + TC_BN_MAX;
            uint32_t it = 0, ygrp = 0, xt = 0;
            TC_PROF_DECL;
            for (int tt = pair; tt < t_end; tt += n_pairs) {
                const int t = tile_of(tt);
                if (t >= p.n_tiles) continue;  // same decision in every role of both CTAs
                if (p.xy == 2) {
                    // cross-first ping-pong (forward GEMMs): the chunks of p.flush stages alternate between the two 256-column
                    // buffers as below, but inside a chunk ALL cross terms are issued before the first hi.hi product: an MMA
                    // adds into its accumulator with truncation, an error of one ulp of the ACCUMULATOR whatever the size of
                    // the addend, so the 2 * 8 cross additions per stage must land while the accumulator is still small; the
                    // large additions per drain are then the hi.hi ones only, as with an accumulator of their own, and two
                    // chunks of run-way remain for the final phase of the previous tile.  p.flush <= NST (host-checked).
                    for (int kb0 = 0; kb0 < nkb; kb0 += p.flush) {
                        const int nst = nkb - kb0 < p.flush ? nkb - kb0 : p.flush;
                        const int a = ygrp & 1;
                        const uint32_t d_tmem = tmem_base + (uint32_t)a * TC_BN_MAX;
                        TC_PROF(2, mbar_wait(bar_tempty(a), ((ygrp >> 1) & 1) ^ 1));
                        tcgen05_fence_after();
                        const uint64_t astep = F16 ? 2 : 64;
                        uint32_t acc = 0u;
                        for (int pass = 0; pass < 2; ++pass) {
                            for (int q = 0; q < nst; ++q) {
                                const uint32_t itq = it + (uint32_t)q;
                                const int s = itq % NST;
                                if (pass == 0) {
                                    TC_PROF(1, mbar_wait(bar_split(s), (itq / NST) & 1));
                                    tcgen05_fence_after();
                                }
                                const int krem = p.K - (kb0 + q) * BK;
                                const int ksteps = krem >= BK ? BK / Cfg::KSTEP : (krem + Cfg::KSTEP - 1) / Cfg::KSTEP;
                                const uint64_t db_hi = make_smem_desc<Cfg::ROWB>(b_hi(s)), db_lo = make_smem_desc<Cfg::ROWB>(b_lo(s));
                                const uint64_t da_hi = F16 ? make_smem_desc<Cfg::ROWB>(a_hi(s)) : make_smem_desc_mn128(a_hi(s), BK * 128);
                                const uint64_t da_lo = F16 ? make_smem_desc<Cfg::ROWB>(a_lo(s)) : make_smem_desc_mn128(a_lo(s), BK * 128);
                                if (pass == 0) {
                                    for (int k = 0; k < ksteps && !(TC_DBG(p) & 2); ++k) {
                                        const uint64_t koff = (uint64_t)(2 * k), aoff = astep * k;
                                        if (F16) {
                                            mma_f16_ss_pair(d_tmem, da_lo + aoff, db_hi + koff, idesc, acc);
                                            mma_f16_ss_pair(d_tmem, da_hi + aoff, db_lo + koff, idesc, 1u);
                                        } else {
                                            mma_tf32_ss_pair(d_tmem, da_lo + aoff, db_hi + koff, idesc, acc);
                                            mma_tf32_ss_pair(d_tmem, da_hi + aoff, db_lo + koff, idesc, 1u);
                                        }
                                        acc = 1u;
                                    }
                                } else {
                                    for (int k = 0; k < ksteps; ++k) {
                                        const uint64_t koff = (uint64_t)(2 * k), aoff = astep * k;
                                        if (F16) mma_f16_ss_pair(d_tmem, da_hi + aoff, db_hi + koff, idesc, acc);
                                        else mma_tf32_ss_pair(d_tmem, da_hi + aoff, db_hi + koff, idesc, acc);
                                        acc = 1u;
                                    }
                                    mma_commit_pair(bar_empty(s), 3);
                                }
                            }
                        }
                        mma_commit_pair(bar_tfull(a), 3);
                        ++ygrp;
                        it += (uint32_t)nst;
                    }
                    continue;
                }
                for (int kb = 0; kb < nkb; ++kb, ++it) {
                    const int pos = kb % p.flush;
                    const bool y_first = pos == 0, y_last = pos == p.flush - 1 || kb == nkb - 1;
                    const int s = it % NST;
                    if (!p.xy) {
                        // ping-pong scheme (backward GEMMs: forces only, chunks of tc_flush_k_bwd): all three products of a
                        // chunk of p.flush stages go to ONE of the two 256-column buffers, which alternate from chunk to
                        // chunk; with two chunks per tile the MMAs of the next tile run through the whole final phase of
                        // this one
                        const int a = ygrp & 1;
                        const uint32_t d_tmem = tmem_base + (uint32_t)a * TC_BN_MAX;
                        if (y_first) {
                            TC_PROF(2, mbar_wait(bar_tempty(a), ((ygrp >> 1) & 1) ^ 1));
                            tcgen05_fence_after();
                        }
                        TC_PROF(1, mbar_wait(bar_split(s), (it / NST) & 1));
                        tcgen05_fence_after();
                        const int krem = p.K - kb * BK;
                        const int ksteps = krem >= BK ? BK / Cfg::KSTEP : (krem + Cfg::KSTEP - 1) / Cfg::KSTEP;
                        const uint64_t db_hi = make_smem_desc<Cfg::ROWB>(b_hi(s)), db_lo = make_smem_desc<Cfg::ROWB>(b_lo(s));
                        const uint64_t da_hi = F16 ? make_smem_desc<Cfg::ROWB>(a_hi(s)) : make_smem_desc_mn128(a_hi(s), BK * 128);
                        const uint64_t da_lo = F16 ? make_smem_desc<Cfg::ROWB>(a_lo(s)) : make_smem_desc_mn128(a_lo(s), BK * 128);
                        const uint64_t astep = F16 ? 2 : 64;
                        uint32_t acc = !y_first;
                        for (int k = 0; k < ksteps && !(TC_DBG(p) & 2); ++k) {  // small cross terms first
                            const uint64_t koff = (uint64_t)(2 * k), aoff = astep * k;
                            if (F16) {
                                mma_f16_ss_pair(d_tmem, da_lo + aoff, db_hi + koff, idesc, acc);
                                mma_f16_ss_pair(d_tmem, da_hi + aoff, db_lo + koff, idesc, 1u);
                            } else {
                                mma_tf32_ss_pair(d_tmem, da_lo + aoff, db_hi + koff, idesc, acc);
                                mma_tf32_ss_pair(d_tmem, da_hi + aoff, db_lo + koff, idesc, 1u);
                            }
                            acc = 1u;
                        }
                        for (int k = 0; k < ksteps; ++k) {
                            const uint64_t koff = (uint64_t)(2 * k), aoff = astep * k;
                            if (F16) mma_f16_ss_pair(d_tmem, da_hi + aoff, db_hi + koff, idesc, acc);
                            else mma_tf32_ss_pair(d_tmem, da_hi + aoff, db_hi + koff, idesc, acc);
                            acc = 1u;
                        }
                        mma_commit_pair(bar_empty(s), 3);
                        if (y_last) {
                            mma_commit_pair(bar_tfull(a), 3);
                            ++ygrp;
                        }
                        continue;
                    }
                    TC_PROF(1, mbar_wait(bar_split(s), (it / NST) & 1));
                    tcgen05_fence_after();
                    const int krem = p.K - kb * BK;
                    const int ksteps = krem >= BK ? BK / Cfg::KSTEP : (krem + Cfg::KSTEP - 1) / Cfg::KSTEP;
                    const uint64_t db_hi = make_smem_desc<Cfg::ROWB>(b_hi(s)), db_lo = make_smem_desc<Cfg::ROWB>(b_lo(s));
                    const uint64_t da_hi = F16 ? make_smem_desc<Cfg::ROWB>(a_hi(s)) : make_smem_desc_mn128(a_hi(s), BK * 128);
                    const uint64_t da_lo = F16 ? make_smem_desc<Cfg::ROWB>(a_lo(s)) : make_smem_desc_mn128(a_lo(s), BK * 128);
                    // per k step: B (and a K-major A) advance 32 bytes along the row, the MN-major A one 1024-byte atom
                    const uint64_t astep = F16 ? 2 : 64;
                    if (kb == 0) {  // X of the previous tile drained by both CTAs
                        TC_PROF(2, mbar_wait(bar_tempty(1), (xt & 1) ^ 1));
                        tcgen05_fence_after();
                    }
                    uint32_t acc = kb != 0;
                    for (int k = 0; k < ksteps && !(TC_DBG(p) & 2); ++k) {
                        const uint64_t koff = (uint64_t)(2 * k), aoff = astep * k;
                        if (F16) {
                            mma_f16_ss_pair(d_x, da_lo + aoff, db_hi + koff, idesc, acc);
                            mma_f16_ss_pair(d_x, da_hi + aoff, db_lo + koff, idesc, 1u);
                        } else {
                            mma_tf32_ss_pair(d_x, da_lo + aoff, db_hi + koff, idesc, acc);
                            mma_tf32_ss_pair(d_x, da_hi + aoff, db_lo + koff, idesc, 1u);
                        }
                        acc = 1u;
                    }
                    if (y_first) {  // Y of the previous group drained (the cross terms above keep the pipe busy meanwhile)
                        TC_PROF(2, mbar_wait(bar_tempty(0), (ygrp & 1) ^ 1));
                        tcgen05_fence_after();
                    }
                    acc = !y_first;
                    for (int k = 0; k < ksteps; ++k) {
                        const uint64_t koff = (uint64_t)(2 * k), aoff = astep * k;
                        if (F16) mma_f16_ss_pair(d_y, da_hi + aoff, db_hi + koff, idesc, acc);
                        else mma_tf32_ss_pair(d_y, da_hi + aoff, db_hi + koff, idesc, acc);
                        acc = 1u;
                    }
                    mma_commit_pair(bar_empty(s), 3);
                    if (y_last) {
                        mma_commit_pair(bar_tfull(0), 3);
                        ++ygrp;
                    }
                    if (kb == nkb - 1) {
                        mma_commit_pair(bar_tfull(1), 3);
                        ++xt;
                    }
                }
            }
            TC_PROF_FLUSH(EPI);
        }
    } else if (warp < TC_FIRST_EPI_WARP) {
        setmaxnreg_dec<Cfg::REGS_SPLIT>();
        // ===== splitters: own A tile into hi and lo (B arrives split: model->Ws / WTs / Wh / WTh) =====
        const int tid = threadIdx.x - TC_FIRST_SPLIT_WARP * 32;
        const float ascale = F16 ? pow2i(14 - amax_exponent(*p.amax_a)) : 1.f;
        uint32_t it = 0;
        TC_PROF_DECL;
        for (int tt = pair; tt < t_end; tt += n_pairs) {
                const int t = tile_of(tt);
                if (t >= p.n_tiles) continue;  // same decision in every role of both CTAs
            for (int kb = 0; kb < nkb; ++kb, ++it) {
                const int s = it % NST;
                TC_PROF(6, mbar_wait(bar_full(s), (it / NST) & 1));
                uint8_t *stage = smem_gen + (size_t)s * Cfg::STAGE_BYTES;
                if (TC_DBG(p) & 1) {
                    if (F16) asm volatile("bar.sync 1, 128;" ::: "memory");
                } else if (F16) {
                    split_f16_tile<BK>(stage, tid, ascale, p.K - kb * BK);
                } else {
                    float4 *ah = reinterpret_cast<float4 *>(stage);
                    split_hi_lo(ah, ah + Cfg::A_BYTES / 16, Cfg::A_BYTES / 16, tid);
                }
                fence_proxy_async_smem();  // own shared memory, read next by the tensor core (async proxy)
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(bar_split(s), 0);
            }
        }
        if (tid == 0) TC_PROF_FLUSH(EPI);
    } else {
        setmaxnreg_inc<Cfg::REGS_EPI>();
        // ===== epilogue: this CTA's 128 rows =====
        const int quad = warp & 3;
        const int half = (warp - TC_FIRST_EPI_WARP) >> 2;
        const int n_groups = (p.bn + 31) / 32;
        const int n_ygroups = (nkb + p.flush - 1) / p.flush;
        const uint32_t lane_base = tmem_base + ((uint32_t)(quad * 32) << 16);
        const int osc_e = F16 ? amax_exponent(*p.amax_a) + amax_exponent(*p.amax_b) - 28 : 0;
        const float oscale = pow2i(osc_e), inv_oscale = pow2i(-osc_e);
        float tmax = 0.f;
        uint32_t ygrp = 0, xt = 0;
        const bool xy = p.xy == 1;  // X / Y accumulators; otherwise chunks alternate between the two buffers
        TC_PROF_DECL;
        for (int tt = pair; tt < t_end; tt += n_pairs) {
                const int t = tile_of(tt);
                if (t >= p.n_tiles) continue;  // same decision in every role of both CTAs
            const int m0 = (2 * (t / p.n_tiles_n) + (int)rank) * TC_BM, n0 = (t % p.n_tiles_n) * p.bn;
            const int row = m0 + quad * 32 + lane;
            const bool row_ok = row < p.M;
            float acc[4][32];
            tc_init_acc<EPI>(p, acc, n0, half, inv_oscale);  // the forward bias rides in the accumulators
            // the hi.hi groups (accumulator Y), then the tile's cross terms (accumulator X): round-to-nearest adds in registers
            for (int c = 0; c < n_ygroups + (xy ? 1 : 0); ++c) {
                // X / Y scheme: buffer 0 = Y (columns 256..511) for the hi.hi groups, then buffer 1 = X (columns 0..255);
                // ping-pong scheme: chunk c sits in buffer (chunk number) & 1 at columns 256 * buffer
                const int a = xy ? (c < n_ygroups ? 0 : 1) : (int)(ygrp & 1);
                TC_PROF(3, mbar_wait(bar_tfull(a), xy ? ((a == 0 ? ygrp : xt) & 1) : ((ygrp >> 1) & 1)));
                tcgen05_fence_after();
                TC_PROF_BEGIN(t_drain);
                const uint32_t col0 = xy ? (a == 0 ? TC_BN_MAX : 0) : (uint32_t)a * TC_BN_MAX;
#pragma unroll
                for (int gi = 0; gi < 4; ++gi) {
                    const int g = 2 * gi + half;
                    if (g < n_groups && !(a == 1 && (TC_DBG(p) & 2)) && !(TC_DBG(p) & 16)) {  // 16: knock-out of the drains
                        uint32_t v[32];
                        tmem_ld_32x32(lane_base + col0 + (uint32_t)(g * 32), v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 32; ++j) acc[gi][j] += __uint_as_float(v[j]);
                    }
                }
                TC_PROF_END(7, t_drain);
                tcgen05_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(bar_tempty(a), 0);
                if (!xy || a == 0) ++ygrp;
                else ++xt;
            }
            TC_PROF_BEGIN(t_final);
            if (EPI == EPI_HIDDEN || EPI == EPI_HIDDEN_HEAD)
                tc_finish_tile<EPI, F16>(p, acc, m0, n0, quad, lane, half, row_ok, oscale, tmax);
            else  // backward: multiplier loads in bursts of 16 ahead of their use
                tc_store_tile<EPI, F16>(p, acc, m0, n0, quad, lane, half, n_groups, row_ok, oscale, tmax);
            TC_PROF_END(4, t_final);
        }
        if (warp == TC_FIRST_EPI_WARP && lane == 0) TC_PROF_FLUSH(EPI);
        if (F16 && p.amax_out && (EPI == EPI_HIDDEN || EPI == EPI_MUL)) {
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
            if (lane == 0) atomicMax(p.amax_out, __float_as_uint(tmax));
        }
    }

    tcgen05_fence_before();
    cluster_sync_all();  // no CTA leaves while its partner may still signal it or read its shared memory
    if (warp == 1) tmem_dealloc_pair<512>(tmem_base);
}

template <bool F16, int BK, int EPI>
static int tc_launch_pair(const CUtensorMap &tmA, const CUtensorMap &tmB, const TcArgs &args, cudaStream_t st) {
    using Cfg = TcPairCfg<F16, BK>;
    static bool attr_on[MAX_DEVICES] = {};
    bool &attr_set = attr_on[current_device()];
    if (!attr_set) {
        GMNN_CUDA(cudaFuncSetAttribute(k_gemm_tc_pair<F16, BK, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        attr_set = true;
    }
    int grid = 2 * args.n_tiles < tc_num_sms() ? 2 * args.n_tiles : (tc_num_sms() & ~1);
    k_gemm_tc_pair<F16, BK, EPI><<<grid, TC_THREADS, Cfg::SMEM_BYTES, st>>>(tmA, tmB, args);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// ---- host side --------------------------------------------------------------------------------

typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode() {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_encodeTiled>(p);
    }
    return fn;
}

// fp32 row-major [rows][K] matrix, box = box_rows x BK elements, swizzle span = BK * 4 bytes.
static int make_tmap(CUtensorMap *tm, const float *base, int64_t rows, int K, int box_rows, int BK) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) {
        set_error("cuTensorMapEncodeTiled is not available from the driver");
        return GMNN_CUDA_ERROR;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)K * 4};
    const cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUtensorMapSwizzle sw = BK == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
    const CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed (%d) for a [%lld][%d] matrix", (int)r, (long long)rows, K);
        return GMNN_CUDA_ERROR;
    }
    return GMNN_OK;
}

static int tc_num_sms() {
    static int n_on[MAX_DEVICES] = {};
    const int dev = current_device();
    int &n = n_on[dev];
    if (!n) {
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (n <= 0) n = 148;
    }
    return n;
}

// Columns per tile: a multiple of 16 (UMMA M = 128 needs N % 16 == 0), at most 256, least padding.
static int pick_bn(int N) {
    if (N <= TC_BN_MAX) return (N + 15) / 16 * 16;
    int best = 256, best_pad = 1 << 30;
    for (int bn = 256; bn >= 128; bn -= 16) {
        const int pad = (N + bn - 1) / bn * bn - N;
        if (pad < best_pad) best_pad = pad, best = bn;
    }
    return best;
}

// Tile-transposed activations [tiles][K][128] as a 2-D tensor of 512-byte lines (line = tile * K + k),
// box {32 floats, BK lines}: four loads per stage give [4][BK][32 floats], the MN-major
// operand layout of make_smem_desc_mn128 (128-byte swizzle, 32-byte atomicity).
static int make_tmap_a(CUtensorMap *tm, const float *base, int64_t M, int K, int BK) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) {
        set_error("cuTensorMapEncodeTiled is not available from the driver");
        return GMNN_CUDA_ERROR;
    }
    const int64_t tiles = (M + TC_BM - 1) / TC_BM;
    const cuuint64_t dims[2] = {(cuuint64_t)TC_BM, (cuuint64_t)(tiles * K)};
    const cuuint64_t strides[1] = {(cuuint64_t)TC_BM * 4};
    const cuuint32_t box[2] = {32, (cuuint32_t)BK};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed (%d) for a tile-transposed [%lld][%d] matrix", (int)r, (long long)M, K);
        return GMNN_CUDA_ERROR;
    }
    return GMNN_OK;
}

template <bool SPLIT, int BK, int EPI>
static int tc_launch(const CUtensorMap &tmA, const CUtensorMap &tmB, const TcArgs &args, cudaStream_t st) {
    using Cfg = TcCfg<SPLIT, BK>;
    static bool attr_on[MAX_DEVICES] = {};
    bool &attr_set = attr_on[current_device()];
    if (!attr_set) {
        GMNN_CUDA(cudaFuncSetAttribute(k_gemm_tc<SPLIT, BK, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        attr_set = true;
    }
    const int grid = args.n_tiles < tc_num_sms() ? args.n_tiles : tc_num_sms();
    k_gemm_tc<SPLIT, BK, EPI><<<grid, TC_THREADS, Cfg::SMEM_BYTES, st>>>(tmA, tmB, args);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int g_tc_pair = 1;    // knob "tc_pair": 3xTF32 GEMMs on CTA pairs (cta_group::2)
int g_tc_dmul_prefetch = 0;  // knob "tc_dmul_prefetch": stages before the last of a tile at which the backward GEMM prefetches its multiplier block (-1: never)
int g_tc_fwd_scheme = 2;  // knob "tc_fwd_scheme": accumulator scheme of the forward GEMMs (TcArgs::xy): 1 or 2
int g_tc_tile_order = 0;  // knob "tc_tile_order": bit 0 forward GEMMs, bit 1 backward GEMMs: column tiles of a row tile back to back on one pair
int g_tc_flush_k_bwd = 256;  // knob "tc_flush_k_bwd": K extent between drains of the hi.hi accumulator, backward GEMMs
#ifdef GMNN_EXPERIMENTS
int g_tc_debug = 0;
}  // namespace gmnn
extern "C" int gmnn_debug_tc_prof(long long *out, int reset) {  // experiments build: [4][160][8] cycle counters
    if (out && cudaMemcpyFromSymbol(out, gmnn::g_tc_prof, sizeof(gmnn::g_tc_prof)) != cudaSuccess) return -1;
    if (reset) {
        static long long zero[4 * 160 * 8] = {};
        if (cudaMemcpyToSymbol(gmnn::g_tc_prof, zero, sizeof(zero)) != cudaSuccess) return -1;
    }
    return 0;
}
namespace gmnn {
#endif
int g_tc_flush_k = 128;  // knob "tc_flush_k": K extent between drains of the hi.hi accumulator, forward GEMMs (CTA pairs)
int g_tc_split_bk = 32;  // knob (gmnn_system_set_int "tc_split_bk"): K extent of a 3xTF32 stage, 16 or 32
int g_tc_h_bk = 64;      // knob "tc_h_bk": K extent of a 3xFP16 stage, 32 or 64

// fp16 row-major [rows][K] matrix (the stacked hi / lo weights), box = box_rows x BK, swizzle span = BK * 2 bytes.
static int make_tmap_h(CUtensorMap *tm, const uint16_t *base, int64_t rows, int K, int box_rows, int BK) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) {
        set_error("cuTensorMapEncodeTiled is not available from the driver");
        return GMNN_CUDA_ERROR;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)K * 2};
    const cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUtensorMapSwizzle sw = BK == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
    const CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<uint16_t *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed (%d) for a fp16 [%lld][%d] matrix", (int)r, (long long)rows, K);
        return GMNN_CUDA_ERROR;
    }
    return GMNN_OK;
}

// Tile-transposed activations as whole [BK][128] fp32 boxes, not swizzled (3xFP16: the splitter warps
// read them, the tensor core does not).
static int make_tmap_a_land(CUtensorMap *tm, const float *base, int64_t M, int K, int BK) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) {
        set_error("cuTensorMapEncodeTiled is not available from the driver");
        return GMNN_CUDA_ERROR;
    }
    const int64_t tiles = (M + TC_BM - 1) / TC_BM;
    const cuuint64_t dims[2] = {(cuuint64_t)TC_BM, (cuuint64_t)(tiles * K)};
    const cuuint64_t strides[1] = {(cuuint64_t)TC_BM * 4};
    const cuuint32_t box[2] = {(cuuint32_t)TC_BM, (cuuint32_t)BK};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled failed (%d) for a tile-transposed [%lld][%d] matrix (fp32 boxes)", (int)r, (long long)M, K);
        return GMNN_CUDA_ERROR;
    }
    return GMNN_OK;
}

// 3xFP16 operands of one GEMM: stacked fp16 hi / lo weights and the absolute-maximum scalars (see TcArgs)
struct TcHalf {
    const uint16_t *Bh = nullptr;
    const uint32_t *amax_a = nullptr, *amax_b = nullptr;
    uint32_t *amax_out = nullptr;
};

// C[M][N] = A[M][K] . Bt[N][K]^T.  A, C, C2, Dmul are tile-transposed ([M/128][cols][128], padded to whole
// tiles); Bt (weights) is row-major [N][K], or for split = true the stacked hi / lo split [2N][K]; with
// `hf` (3xFP16, always on CTA pairs) the fp16 split hf->Bh replaces Bt.
int tc_gemm(bool split, int epi, int64_t M, int N, int K, const float *A, const float *Bt, float *C, const float *bias,
            float *C2, const float *Dmul, cudaStream_t st, const float *w_head = nullptr, float *ypart = nullptr,
            int *n_slots = nullptr, const TcHalf *hf = nullptr, int64_t m_pad_total = 0, int dmul_N = 0, int dmul_row_div = 1) {
    if (K % 8 != 0 || N % 8 != 0 || M <= 0 || M > INT32_MAX) {
        set_error("tensor-core MLP: widths must be multiples of 8 (K = %d, N = %d)", K, N);
        return GMNN_UNSUPPORTED;
    }
    const int BK = hf ? g_tc_h_bk : (split ? g_tc_split_bk : 32);
    TcArgs a = {};
    a.M = (int)M, a.N = N, a.K = K;
    a.bn = pick_bn(N);
    a.n_tiles_n = (N + a.bn - 1) / a.bn;
    a.n_tiles = (int)((M + TC_BM - 1) / TC_BM) * a.n_tiles_n;
    // Accumulator flushes (the tensor core adds into its fp32 accumulator with truncation):
    //   CTA-pair kernels: the hi.hi accumulator is drained every tc_flush_k of K on the forward GEMMs (they enter the
    //     energies) and every tc_flush_k_bwd on the backward GEMMs (forces only: error budget 1e-4); the cross terms have
    //     an accumulator of their own that lasts the whole tile;
    //   single-CTA kernel (tc_pair = 0, and the single-pass TF32 mode: one chunk): mixed accumulator, every 64 of K.
    const bool fwd = epi == EPI_HIDDEN || epi == EPI_HIDDEN_HEAD;
    const bool pair_kernel = hf != nullptr || (split && g_tc_pair);
    const int flush_k = pair_kernel ? (fwd ? g_tc_flush_k : g_tc_flush_k_bwd) : 64;
    a.flush = split ? (flush_k / BK > 0 ? flush_k / BK : 1) : (K + BK - 1) / BK;
    a.flush1 = a.flush;
    a.dmul_pf = g_tc_dmul_prefetch;
    a.xy = fwd ? g_tc_fwd_scheme : 0;
    {  // scheme 2 holds a whole chunk in the stage ring
        const int es = hf ? 2 : 4, n_stages = TC_STAGE_BYTES_TOTAL / (2 * (TC_BM * BK * es + (TC_BN_MAX / 2) * BK * es));
        if (a.xy == 2 && a.flush > n_stages) a.xy = 1;
    }
    a.order = (g_tc_tile_order >> (fwd ? 0 : 1)) & 1;
#ifdef GMNN_EXPERIMENTS
    a.debug = g_tc_debug;
#else
    a.debug = 0;
#endif
    a.C = C, a.C2 = C2, a.bias = bias, a.Dmul = Dmul;
    a.dmul_N = dmul_N > 0 ? dmul_N : N, a.dmul_row_div = dmul_row_div > 0 ? dmul_row_div : 1;
    // ypart is [slots][m_pad]: with row segments the caller hands ypart + row0 and the padded row count of the whole matrix
    a.w_head = w_head, a.ypart = ypart, a.m_pad = m_pad_total > 0 ? m_pad_total : (M + TC_BM - 1) / TC_BM * TC_BM;
    a.amax_a = hf ? hf->amax_a : nullptr, a.amax_b = hf ? hf->amax_b : nullptr, a.amax_out = hf ? hf->amax_out : nullptr;
    if (n_slots) *n_slots = 2 * a.n_tiles_n;
    CUtensorMap tmA, tmB;
    int rc;
#define TC_PAIR_CASE(F16V, BKV)                                                                       \
    switch (epi) {                                                                                    \
        case EPI_PLAIN: return tc_launch_pair<F16V, BKV, EPI_PLAIN>(tmA, tmB, a, st);                  \
        case EPI_HIDDEN: return tc_launch_pair<F16V, BKV, EPI_HIDDEN>(tmA, tmB, a, st);                \
        case EPI_HIDDEN_HEAD: return tc_launch_pair<F16V, BKV, EPI_HIDDEN_HEAD>(tmA, tmB, a, st);      \
        default: return tc_launch_pair<F16V, BKV, EPI_MUL>(tmA, tmB, a, st);                           \
    }
    if (hf) {
        a.n_tiles = (int)(((M + TC_BM - 1) / TC_BM + 1) / 2) * a.n_tiles_n;
        if ((rc = make_tmap_a_land(&tmA, A, M, K, BK))) return rc;
        if ((rc = make_tmap_h(&tmB, hf->Bh, 2 * (int64_t)N, K, a.bn / 2, BK))) return rc;
        if (BK == 64) { TC_PAIR_CASE(true, 64) }
        TC_PAIR_CASE(true, 32)
    }
    if ((rc = make_tmap_a(&tmA, A, M, K, BK))) return rc;
    if ((rc = make_tmap(&tmB, Bt, split ? 2 * (int64_t)N : N, K, a.bn, BK))) return rc;
#define TC_CASE(SP, BKV)                                                                  \
    switch (epi) {                                                                        \
        case EPI_PLAIN: return tc_launch<SP, BKV, EPI_PLAIN>(tmA, tmB, a, st);             \
        case EPI_HIDDEN: return tc_launch<SP, BKV, EPI_HIDDEN>(tmA, tmB, a, st);           \
        case EPI_HIDDEN_HEAD: return tc_launch<SP, BKV, EPI_HIDDEN_HEAD>(tmA, tmB, a, st); \
        default: return tc_launch<SP, BKV, EPI_MUL>(tmA, tmB, a, st);                      \
    }
    if (split && g_tc_pair) {
        // pair tiles: two adjacent 128-row tiles x one column tile; B box = this CTA's half of the columns
        a.n_tiles = (int)(((M + TC_BM - 1) / TC_BM + 1) / 2) * a.n_tiles_n;
        if ((rc = make_tmap(&tmB, Bt, 2 * (int64_t)N, K, a.bn / 2, BK))) return rc;
        if (BK == 32) { TC_PAIR_CASE(false, 32) }
        TC_PAIR_CASE(false, 16)
    }
    if (!split) { TC_CASE(false, 32) }
    if (BK == 32) { TC_CASE(true, 32) }
    TC_CASE(true, 16)
#undef TC_CASE
#undef TC_PAIR_CASE
}

// ---- operand preparation ----------------------------------------------------------------------
__global__ void k_absmax(const float *__restrict__ src, int64_t n, uint32_t *__restrict__ amax) {
    float m = 0.f;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x)
        m = fmaxf(m, fabsf(src[t]));
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(amax, __float_as_uint(m));
}

// dst[0, n) = fp16(src * 2^s), dst[n, 2n) = fp16(src * 2^s - hi), 2^s from *amax (the 3xFP16 B operand)
__global__ void k_split_stack_h(const float *__restrict__ src, __half *__restrict__ dst, int64_t n,
                                const uint32_t *__restrict__ amax) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= n) return;
    const float v = src[t] * pow2i(14 - amax_exponent(*amax));
    const __half h = __float2half_rn(v);
    dst[t] = h;
    dst[n + t] = __float2half_rn(v - __half2float(h));
}

// *amax = max |src| (reset first)
int launch_absmax(const float *src, int64_t n, uint32_t *amax, cudaStream_t st) {
    GMNN_CUDA(cudaMemsetAsync(amax, 0, sizeof(uint32_t), st));
    k_absmax<<<(unsigned)((n + 1023) / 1024 < 256 ? (n + 1023) / 1024 : 256), 256, 0, st>>>(src, n, amax);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// the stacked fp16 split of src scaled by the power of two that *amax (>= max |src|) fixes
int launch_split_stack_h(const float *src, uint16_t *dst, int64_t n, const uint32_t *amax, cudaStream_t st) {
    k_split_stack_h<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, reinterpret_cast<__half *>(dst), n, amax);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

__global__ void k_split_stack(const float *__restrict__ src, float *__restrict__ dst, int64_t n) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= n) return;
    const float v = src[t], h = to_tf32_rna(v);
    dst[t] = h;
    dst[n + t] = v - h;
}

int launch_split_stack(const float *src, float *dst, int64_t n, cudaStream_t st) {
    k_split_stack<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, dst, n);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_mlp_forward_tc(gmnn_system *s, cudaStream_t st) {
    const gmnn_model *m = s->model;
    const bool f16 = s->mlp_precision == GMNN_MLP_3XF16;
    const bool split = s->mlp_precision == GMNN_MLP_3XTF32 || f16;
    MlpSeg seg[MAX_SPECIES];
    const int ns = mlp_segments(s, seg);
    const int64_t m_pad = (s->n_rows + TC_BM - 1) / TC_BM * TC_BM;
    const float *X = s->G;
    for (int l = 0; l < m->hp.n_hidden; ++l) {
        // z = X W[l]: the B operand is W[l]^T = WT[l], [fan_out][fan_in]
        // single head: the last hidden layer's epilogue takes the head's dot product itself
        const int fi = m->dims[l], fo = m->dims[l + 1];
        const bool fuse = l == m->hp.n_hidden - 1 && (m->hp.n_heads == 1 || s->use_mean_head) && 2 * ((fo + 127) / 128) <= MAX_HEAD_SLOTS;
        s->heads_fused = fuse;
        for (int q = 0; q < ns; ++q) {  // layer-major: every segment of layer l before layer l + 1 (operand maxima)
            const int64_t r0 = seg[q].row0;
            const int t = seg[q].set;
            const size_t ws = m->wsize(l);
            TcHalf hf;
            hf.Bh = m->WTh[l] + 2 * t * ws, hf.amax_b = m->wmax + l;
            hf.amax_a = s->amax + (l == 0 ? AMAX_G : AMAX_H + l - 1), hf.amax_out = s->amax + AMAX_H + l;
            const float *w_head = (fuse && s->use_mean_head) ? m->w_mean + (size_t)t * (fo + 1) : m->W[l + 1] + t * m->wsize(l + 1);
            int rc = tc_gemm(split, fuse ? EPI_HIDDEN_HEAD : EPI_HIDDEN, seg[q].rows, fo, fi, tile_rows(X, r0, fi),
                             split ? m->WTs[l] + 2 * t * ws : m->WT[l] + t * ws, tile_rows(s->H[l], r0, fo),
                             m->b[l] + (size_t)t * fo, tile_rows(s->D[l], r0, fo), nullptr, st, w_head, s->ypart + r0,
                             &s->head_slots, f16 ? &hf : nullptr, m_pad);
            if (rc) return rc;
        }
        X = s->H[l];
    }
    return GMNN_OK;
}

// Same chain as launch_mlp_backward_simt (mlp_simt.cu); the B operand of  out = Aop . Bop  is Bop^T:
// Bop = WT[l-1] gives W[l-1]; Bop = diag(v) WT[L-1] gives W[L-1] diag(v) = BvT.
int launch_mlp_backward_tc(gmnn_system *s, const float *head_w_dev, cudaStream_t st) {
    const gmnn_model *m = s->model;
    const bool f16 = s->mlp_precision == GMNN_MLP_3XF16;
    const bool split = s->mlp_precision == GMNN_MLP_3XTF32 || f16;
    const int L = m->hp.n_hidden;
    int rc = GMNN_OK;
    const size_t nbv = (size_t)m->dims[L] * m->dims[L - 1];
    // The seeded operand W[L-1] diag(W_last c), its maximum and its split depend on the head weights c only: for the
    // model's constant mean-head weights (every gmnn_energy_forces call and MD step) they are prepared once and kept
    // (4 - 5 small launches less per evaluation: 15 % of the launches of a step); any other c (one-hot ensemble heads,
    // UDD weights) prepares them anew.  Dropped by any gmnn_system_set_int and by the batched ensemble pass.
    const bool keep = head_w_dev == m->head_mean_w;
    if (!(keep && s->seed_w == head_w_dev && s->seed_prec == s->mlp_precision)) {
        s->seed_w = nullptr;
        if ((rc = launch_mlp_seed(s, head_w_dev, st))) return rc;  // vhead, BvT per weight set (see mlp_simt.cu)
        if (f16) {  // one scale for the seeded operands of all sets
            if ((rc = launch_absmax(s->BvT, (int64_t)(nbv * m->n_sets), s->amax + AMAX_BVT, st))) return rc;
            for (int t = 0; t < m->n_sets; ++t)
                if ((rc = launch_split_stack_h(s->BvT + t * nbv, s->BvTh + 2 * t * nbv, (int64_t)nbv, s->amax + AMAX_BVT, st))) return rc;
        } else if (split) {
            for (int t = 0; t < m->n_sets; ++t)
                if ((rc = launch_split_stack(s->BvT + t * nbv, s->BvTs + 2 * t * nbv, (int64_t)nbv, st))) return rc;
        }
        if (keep) s->seed_w = head_w_dev, s->seed_prec = s->mlp_precision;
    }
    MlpSeg seg[MAX_SPECIES];
    const int ns = mlp_segments(s, seg);
    const float *Aop = s->D[L - 1];
    int cur = 0;
    for (int l = L - 1; l >= 0; --l) {
        const int fo = m->dims[l], fi = m->dims[l + 1];  // out = Aop [rows][fi] . Bop [fi][fo]
        const size_t ws = m->wsize(l);
        for (int q = 0; q < ns; ++q) {
            const int64_t r0 = seg[q].row0;
            const int t = seg[q].set;
            const bool seeded = l == L - 1;  // B operand: W[L-1] diag(v) of this set, then the plain W[l]
            const float *BopT = seeded ? (split ? s->BvTs + 2 * t * ws : s->BvT + t * ws) : (split ? m->Ws[l] + 2 * t * ws : m->W[l] + t * ws);
            TcHalf hf;
            hf.Bh = seeded ? s->BvTh + 2 * t * ws : m->Wh[l] + 2 * t * ws;
            hf.amax_b = seeded ? s->amax + AMAX_BVT : m->wmax + l;
            hf.amax_a = seeded ? s->amax + AMAX_D : s->amax + AMAX_DZ + (cur ^ 1);  // swish' of the last hidden layer, then dZ
            if (l > 0) {
                hf.amax_out = s->amax + AMAX_DZ + cur;
                rc = tc_gemm(split, EPI_MUL, seg[q].rows, fo, fi, tile_rows(Aop, r0, fi), BopT, tile_rows(s->dZ[cur], r0, fo),
                             nullptr, nullptr, tile_rows(s->D[l - 1], r0, fo), st, nullptr, nullptr, nullptr, f16 ? &hf : nullptr);
            } else {
                hf.amax_out = nullptr;
                rc = tc_gemm(split, EPI_PLAIN, seg[q].rows, fo, fi, tile_rows(Aop, r0, fi), BopT, tile_rows(s->dG, r0, fo), nullptr,
                             nullptr, nullptr, st, nullptr, nullptr, nullptr, f16 ? &hf : nullptr);
            }
            if (rc) return rc;
        }
        if (l > 0) {
            Aop = s->dZ[cur];
            cur ^= 1;
        }
    }
    return GMNN_OK;
}


// ---- batched shallow-ensemble backward (a12; Eq. 5, 6) -------------------------------------------------
// The backward of head m differs from that of any other head only in the seed v_m = W_last[:, m].  For HB heads at once:
//   first GEMM  (seeded): dZ[rows][HB x w] = D_last[rows][Hd] . [B_0 | B_1 | ... ]^T-stacked, B_m = W[L-1] diag(v_m), one wide
//               GEMM whose column block m is head m (its swish' multiplier is read with column c % w);
//   its output, tile-transposed [row tile][HB x w][128], IS a matrix of HB x as many row tiles of width w, ordered
//               [atom tile][head]: the GEMMs below it run on those stacked rows with the shared weights, and so does the
//               contraction backward (descriptor.cu, `heads`); the pair backward of head m reads rows [tile][m] (a_heads).
// 32 heads x 8 192 atoms become GEMMs of 16 384 columns / 262 144 rows that fill the machine, instead of 32 under-filled ones.
__global__ void k_seed_heads(int prev, int Hd, const float *__restrict__ W, const float *__restrict__ Wlast, int M, int head0,
                             int HB, float *__restrict__ out) {
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;  // out[m][n][k] = W[n][k] Wlast[k][head0 + m]
    const int64_t per = (int64_t)prev * Hd;
    if (t >= per * HB) return;
    const int m = (int)(t / per);
    const int k = (int)(t % Hd);
    out[t] = __ldg(&W[t % per]) * __ldg(&Wlast[(int64_t)k * M + head0 + m]);
}

int launch_mlp_backward_tc_heads(gmnn_system *s, int head0, int HB, cudaStream_t st) {
    const gmnn_model *m = s->model;
    const bool f16 = s->mlp_precision == GMNN_MLP_3XF16;
    const int L = m->hp.n_hidden, M = m->hp.n_heads;
    const int Hd = m->dims[L], prev = m->dims[L - 1];
    const int64_t nbv = (int64_t)prev * Hd * HB;
    int rc;
    s->seed_w = nullptr;  // the batch's maximum goes to the scale word of the kept single-head seed
    k_seed_heads<<<(unsigned)((nbv + 255) / 256), 256, 0, st>>>(prev, Hd, m->W[L - 1], m->W[L], M, head0, HB, s->ens_BvT);
    GMNN_LAUNCHED();
    if (f16) {
        if ((rc = launch_absmax(s->ens_BvT, nbv, s->amax + AMAX_BVT, st))) return rc;
        if ((rc = launch_split_stack_h(s->ens_BvT, s->ens_BvTh, nbv, s->amax + AMAX_BVT, st))) return rc;
    } else if ((rc = launch_split_stack(s->ens_BvT, s->ens_BvTs, nbv, st))) {
        return rc;
    }
    const int64_t rows = s->N, row_tiles = (rows + TC_BM - 1) / TC_BM;
    const float *Aop = s->D[L - 1];
    int cur = 0;
    for (int l = L - 1; l >= 0; --l) {
        const int fo = m->dims[l], fi = m->dims[l + 1];
        const bool seeded = l == L - 1;
        // seeded: [rows] x [HB fo] = [rows][fi] . stacked seeds; below: [row_tiles HB 128] x [fo] with the shared W[l]
        const int64_t Mrows = seeded ? rows : row_tiles * HB * TC_BM;
        const int Ncols = seeded ? HB * fo : fo;
        TcHalf hf;
        hf.Bh = seeded ? s->ens_BvTh : m->Wh[l];
        hf.amax_b = seeded ? s->amax + AMAX_BVT : m->wmax + l;
        hf.amax_a = seeded ? s->amax + AMAX_D : s->amax + AMAX_DZ + (cur ^ 1);
        const float *BopT = seeded ? s->ens_BvTs : m->Ws[l];
        if (l > 0) {
            hf.amax_out = s->amax + AMAX_DZ + cur;
            rc = tc_gemm(true, EPI_MUL, Mrows, Ncols, fi, Aop, BopT, s->ens_dZ[cur], nullptr, nullptr, s->D[l - 1], st, nullptr, nullptr,
                         nullptr, f16 ? &hf : nullptr, 0, fo, seeded ? 1 : HB);
            Aop = s->ens_dZ[cur];
            cur ^= 1;
        } else {
            hf.amax_out = nullptr;
            rc = tc_gemm(true, EPI_PLAIN, Mrows, Ncols, fi, Aop, BopT, s->ens_dG, nullptr, nullptr, nullptr, st, nullptr, nullptr, nullptr,
                         f16 ? &hf : nullptr);
        }
        if (rc) return rc;
    }
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

}  // namespace gmnn
