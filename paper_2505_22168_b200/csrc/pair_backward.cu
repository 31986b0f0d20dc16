// pair_backward.cu -- a10 + a11: the per-pair gradient g_ij = dE/dd_ij and the deterministic force reduction
// F_i = sum_j (g_ij - g_ji)   (virial: SURVEY 8(f) NEXT-3).
//
// Per-pair polynomial: E gets sum_s R_s(r) p_s(u) from pair (i,j), p_s(u) = sum_m A_i[s][m] mono_m(u), so
// g_ij = dE/dd = (sum_s R'_s p_s) u + (grad_u q - (u.grad_u q) u) / r with q(u) = sum_m (sum_s R_s A[s][m]) mono_m(u).
//
// Force reduction, two forms, both without atomics, in a fixed summation order, bit-reproducible
// (the full list is symmetric, (i,j,n) <-> (j,i,-n)):
//   pair buffer (GMNN_FORCE_PAIRBUF, what bench.py times): g_ij is evaluated once per directed pair with
//     the centre's own adjoint A_i and stored into the row of j at the slot of the reverse pair (index
//     built with the list, neighbor.cu); k_force_reduce subtracts each atom's received row in slot order;
//   gather form (GMNN_FORCE_GATHER): each centre evaluates both directions itself, g_ij with A_i and
//     g_ji with the neighbour's A_j (a 400-byte read served by L1/L2).
#include "pair_common.cuh"

namespace gmnn {

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
// GENERAL = false: the configs' model (Gaussian basis, no ZBL, no virial).  GENERAL = true: run-time switches for the
// Bessel-like basis and the ZBL term, and with vir_atom != nullptr the kernel also leaves vir_atom[c][i] = -sum_j d_a g_b
// (c = 3 a + b) over the centre's own directed pairs, whose sum over the atoms is the virial W = -sum_pairs d (x) g =
// -dE/d strain (oracle O-16).
template <int NR, int NB, int LPA, bool PAIRBUF, bool GENERAL>
__global__ void __launch_bounds__(128)
k_pair_backward(int64_t N, const float4 *__restrict__ pos4, const uint32_t *__restrict__ nbr,
                const int32_t *__restrict__ count, int cap, Geometry geo, RadialParams rp,
                const float *__restrict__ beta, const float *__restrict__ A, float *__restrict__ f_int,
                const uint16_t *__restrict__ rev, float4 *__restrict__ gbuf, const int32_t *__restrict__ mrow,
                float *__restrict__ vir_atom, int a_heads, int a_head) {
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
            // row of the adjoint: species-grouped rows (mrow), or head a_head of the batched ensemble buffers
            // ([atom tile][head][128] rows, gmnn_api.cu), else the atom itself
            const int64_t ra = a_heads > 1 ? ((ia >> 7) * a_heads + a_head) * 128 + (ia & 127) : ((mrow && ia < N) ? (int64_t)mrow[ia] : ia);
            s_A[q] = ia < N ? __ldg(&src[ra * (NR * PSI / 4) + q % (NR * PSI / 4)]) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    __syncthreads();
    float fx = 0.f, fy = 0.f, fz = 0.f;
    const bool VIRIAL = GENERAL && vir_atom != nullptr;
    float vir[GENERAL ? 9 : 1];
#pragma unroll
    for (int c = 0; c < (GENERAL ? 9 : 1); ++c) vir[c] = 0.f;
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
                    radial_basis<NB, true, GENERAL>(rp, r, rinv, phi, dphi, fc, dfc);
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
                            const int64_t rj = a_heads > 1 ? (((int64_t)pg.j >> 7) * a_heads + a_head) * 128 + (pg.j & 127)
                                                           : (int64_t)(mrow ? mrow[pg.j] : pg.j);
                            const float4 *Aj = reinterpret_cast<const float4 *>(A) + rj * (NR * PSI / 4);
                            float mono_r[PSI];  // the neighbour sees the bond reversed
                            monomials(-ux, -uy, -uz, mono_r);
                            float hx, hy, hz;  // gradient with respect to (-u): g_ji in the frame of d_ji = -d_ij
                            pair_gradient<NR>([&](int s, int qq) { return __ldg(&Aj[s * (PSI / 4) + qq]); }, R, dR, mono_r,
                                              -ux, -uy, -uz, rinv, hx, hy, hz);
                            gxr = hx, gyr = hy, gzr = hz;
                        }
                    }
                    if (GENERAL && rp.zbl_on && pg.r2 < rp.zbl_r_max2) {  // ZBL: g += d(V/2)/dr u in both directions of the pair
                        float e, de;
                        zbl_half<true>(rp, zi, pg.zj, r, rinv, e, de);
                        gxo = fmaf(de, ux, gxo), gyo = fmaf(de, uy, gyo), gzo = fmaf(de, uz, gzo);
                        if (!PAIRBUF) gxr = fmaf(-de, ux, gxr), gyr = fmaf(-de, uy, gyr), gzr = fmaf(-de, uz, gzr);
                    }
                    if (PAIRBUF) *slot = make_float4(gxo, gyo, gzo, 0.f);
                    if (GENERAL) {
                        if (VIRIAL) {
                            const float dv[3] = {pg.dx, pg.dy, pg.dz}, gv[3] = {gxo, gyo, gzo};
#pragma unroll
                            for (int a = 0; a < 3; ++a)
#pragma unroll
                                for (int b = 0; b < 3; ++b) vir[3 * a + b] = fmaf(-dv[a], gv[b], vir[3 * a + b]);
                        }
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
    if (GENERAL && VIRIAL) {
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
// WELFORD (shallow-ensemble pass, a12): the force of this head is not stored but goes straight into the running
// mean / sum of squared deviations over the heads, at the caller's index perm[i] (Eq. 5: means first, then squared
// deviations; same arithmetic as k_welford on the scattered forces, so the statistics are bit-identical).
__device__ __forceinline__ void welford_update(int head, float v, float *mean, float *m2) {
    if (head == 0) {
        *mean = v;
        *m2 = 0.f;
    } else {
        const float mu = *mean;
        const float d = v - mu;
        const float mu2 = mu + d / (float)(head + 1);
        *mean = mu2;
        *m2 = fmaf(d, v - mu2, *m2);
    }
}

template <int LPA, bool WELFORD>
__global__ void __launch_bounds__(256)
k_force_reduce(int64_t N, const int32_t *__restrict__ count, int cap, const float4 *__restrict__ gbuf,
               float *__restrict__ f_int, const int32_t *__restrict__ perm, int head, float *__restrict__ f_mean,
               float *__restrict__ f_m2) {
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
        if (WELFORD) {
            const int64_t c = perm[i];
            welford_update(head, f_int[3 * i] - fx, f_mean + 3 * c, f_m2 + 3 * c);
            welford_update(head, f_int[3 * i + 1] - fy, f_mean + 3 * c + 1, f_m2 + 3 * c + 1);
            welford_update(head, f_int[3 * i + 2] - fz, f_mean + 3 * c + 2, f_m2 + 3 * c + 2);
        } else {
            f_int[3 * i] -= fx;
            f_int[3 * i + 1] -= fy;
            f_int[3 * i + 2] -= fz;
        }
    }
}

// gather form: the complete force of this head is in f_int; the Welford update alone
__global__ void __launch_bounds__(256)
k_welford_perm(int64_t N, const float *__restrict__ f_int, const int32_t *__restrict__ perm, int head,
               float *__restrict__ f_mean, float *__restrict__ f_m2) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t c = perm[i];
#pragma unroll
    for (int a = 0; a < 3; ++a) welford_update(head, f_int[3 * i + a], f_mean + 3 * c + a, f_m2 + 3 * c + a);
}

// ---------------------------------------------------------------------------------------------
// a12, pair-buffer form, several heads per launch (batched shallow-ensemble pass, gmnn_api.cu ensemble_pass).
// The geometry of a pair, its radial functions R_s, R'_s and the 20 monomials do not depend on the head: they are
// evaluated once per pair and chunk of HC heads (blockIdx.y = chunk), and only the gradient polynomial runs per head with
// that head's adjoint A^(m)_i (rows [atom tile][head][128] of ens_A, staged in shared memory: HC x 400 bytes per centre).
// Head m's own-direction sums go to f_h[m][3 N], its g_ij into gbuf_h[m][N cap]: the same values and the same summation
// order as k_pair_backward<PAIRBUF> launched once per head.
// ---------------------------------------------------------------------------------------------
constexpr int PB_HC = 8;  // heads per chunk at most

template <int NR, int NB, int LPA, bool GENERAL>
__global__ void __launch_bounds__(128)
k_pair_backward_heads(int64_t N, const float4 *__restrict__ pos4, const uint32_t *__restrict__ nbr,
                      const int32_t *__restrict__ count, int cap, Geometry geo, RadialParams rp,
                      const float *__restrict__ beta, const float *__restrict__ A, float *__restrict__ f_h,
                      const uint16_t *__restrict__ rev, float4 *__restrict__ gbuf_h, int a_heads, int hc_max) {
    constexpr int KB = (NB + 3) & ~3;
    constexpr int ROW = NR * KB;
    constexpr int GROUPS = 128 / LPA;
    constexpr int AQ = NR * PSI / 4;  // float4 per adjoint row
    extern __shared__ float s_mem[];
    float *s_beta = s_mem;
    float4 *s_A = reinterpret_cast<float4 *>(s_mem + ((rp.n_species * rp.n_species * ROW + 3) & ~3));
    for (int q = threadIdx.x; q < rp.n_species * rp.n_species * ROW; q += blockDim.x) s_beta[q] = beta[q];
    const int head0 = blockIdx.y * hc_max;
    const int hc = a_heads - head0 < hc_max ? a_heads - head0 : hc_max;
    const int64_t gt = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t i = gt / LPA;
    const int sub = (int)(gt % LPA);
    const int grp = threadIdx.x / LPA;
    const bool live = i < N;
    {  // stage A^(m)_i of the block's centres and the chunk's heads: [group][head][AQ]
        const int64_t first = blockIdx.x * (int64_t)GROUPS;
        const float4 *src = reinterpret_cast<const float4 *>(A);
        for (int q = threadIdx.x; q < GROUPS * hc * AQ; q += blockDim.x) {
            const int g = q / (hc * AQ), h = (q / AQ) % hc, e = q % AQ;
            const int64_t ia = first + g;
            const int64_t ra = ((ia >> 7) * a_heads + head0 + h) * 128 + (ia & 127);
            s_A[(g * hc_max + h) * AQ + e] = ia < N ? __ldg(&src[ra * AQ + e]) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    __syncthreads();
    // own-direction force sums of this thread, one triple per head of the chunk, in shared memory ([head][component][thread]:
    // conflict-free), so that the head loop below stays rolled (one instance of the gradient polynomial in the code)
    float *s_f = reinterpret_cast<float *>(s_A + GROUPS * hc_max * AQ);
    for (int q = 0; q < 3 * hc; ++q) s_f[q * 128 + threadIdx.x] = 0.f;
    if (live) {
        const float4 xi = pos4[i];
        const int zi = __float_as_int(xi.w);
        const int cnt = count[i];
        const uint4 *row = reinterpret_cast<const uint4 *>(nbr + i * (int64_t)cap);
        const uint2 *rrow = reinterpret_cast<const uint2 *>(rev + i * (int64_t)cap);
        const float4 *Ai = s_A + grp * hc_max * AQ;
        const int64_t hstride = N * (int64_t)cap;  // float4 per head in gbuf_h
        uint4 e_next = make_uint4(0u, 0u, 0u, 0u);
        uint2 r_next = make_uint2(0u, 0u);
        if (sub * 4 < cnt) {
            e_next = __ldg(&row[sub]);
            r_next = __ldg(&rrow[sub]);
        }
        for (int k4 = sub; k4 * 4 < cnt; k4 += LPA) {
            const uint4 e4 = e_next;
            const uint2 r2 = r_next;
            if ((k4 + LPA) * 4 < cnt) {
                e_next = __ldg(&row[k4 + LPA]);
                r_next = __ldg(&rrow[k4 + LPA]);
            }
#pragma unroll 1
            for (int q = 0; q < 4; ++q) {
                if (k4 * 4 + q >= cnt) break;
                const uint32_t ent = q == 0 ? e4.x : q == 1 ? e4.y : q == 2 ? e4.z : e4.w;
                const uint32_t rv = ((q < 2 ? r2.x : r2.y) >> ((q & 1) * 16)) & 0xFFFFu;
                const PairGeom pg = pair_geometry(ent, xi, pos4, geo);
                if (rv == 0xFFFFu) continue;  // no partner (overflowed rebuild): flagged by k_build_rev
                float4 *slot = gbuf_h + (int64_t)head0 * hstride + (int64_t)pg.j * cap + rv;
                if (pg.r2 >= rp.r_cut2) {  // skin shell
                    for (int h = 0; h < hc; ++h) slot[h * hstride] = make_float4(0.f, 0.f, 0.f, 0.f);
                    continue;
                }
                const float rinv = rsqrtf(pg.r2);
                const float r = pg.r2 * rinv;
                float phi[NB], dphi[NB], fc, dfc;
                radial_basis<NB, true, GENERAL>(rp, r, rinv, phi, dphi, fc, dfc);
                const float ux = pg.dx * rinv, uy = pg.dy * rinv, uz = pg.dz * rinv;
                float mono[PSI];
                monomials(ux, uy, uz, mono);
                const float4 *bt = reinterpret_cast<const float4 *>(s_beta + (zi * rp.n_species + pg.zj) * ROW);
                float R[NR], dR[NR];
#pragma unroll
                for (int s = 0; s < NR; ++s) {
                    float2 sd = make_float2(0.f, 0.f);
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
                float de = 0.f;
                if (GENERAL && rp.zbl_on && pg.r2 < rp.zbl_r_max2) {  // ZBL: the same term in every head
                    float e;
                    zbl_half<true>(rp, zi, pg.zj, r, rinv, e, de);
                }
#pragma unroll 1
                for (int h = 0; h < hc; ++h) {
                    const float4 *Ah = Ai + h * AQ;
                    float gx, gy, gz;
                    pair_gradient<NR>([&](int s, int qq) { return Ah[s * (PSI / 4) + qq]; }, R, dR, mono, ux, uy, uz, rinv,
                                      gx, gy, gz);
                    if (GENERAL) gx = fmaf(de, ux, gx), gy = fmaf(de, uy, gy), gz = fmaf(de, uz, gz);
                    slot[h * hstride] = make_float4(gx, gy, gz, 0.f);
                    float *f = s_f + (3 * h) * 128 + threadIdx.x;
                    f[0] += gx, f[128] += gy, f[256] += gz;
                }
            }
        }
    }
    for (int h = 0; h < hc; ++h) {
        float fx = s_f[(3 * h) * 128 + threadIdx.x], fy = s_f[(3 * h + 1) * 128 + threadIdx.x], fz = s_f[(3 * h + 2) * 128 + threadIdx.x];
#pragma unroll
        for (int o = LPA / 2; o >= 1; o >>= 1) {
            fx += __shfl_xor_sync(0xffffffffu, fx, o);
            fy += __shfl_xor_sync(0xffffffffu, fy, o);
            fz += __shfl_xor_sync(0xffffffffu, fz, o);
        }
        if (live && sub == 0) {
            float *f = f_h + (int64_t)(head0 + h) * 3 * N + 3 * i;
            f[0] = fx, f[1] = fy, f[2] = fz;
        }
    }
}

// Force of every head of the batch (f_h[m] minus the received row of gbuf_h[m], summed as in k_force_reduce), folded into
// the running statistics over the heads in head order (Eq. 5; welford_update as in the head-by-head path).
template <int LPA>
__global__ void __launch_bounds__(256)
k_force_reduce_heads(int64_t N, const int32_t *__restrict__ count, int cap, const float4 *__restrict__ gbuf_h,
                     const float *__restrict__ f_h, const int32_t *__restrict__ perm, int head_first, int n_heads,
                     float *__restrict__ f_mean, float *__restrict__ f_m2) {
    const int64_t gt = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t i = gt / LPA;
    const int sub = (int)(gt % LPA);
    const int cnt = i < N ? count[i] : 0;
    const int64_t hstride = N * (int64_t)cap;
    for (int h = 0; h < n_heads; ++h) {
        float fx = 0.f, fy = 0.f, fz = 0.f;
        if (i < N) {
            const float4 *row = gbuf_h + h * hstride + i * (int64_t)cap;
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
            const int64_t c = perm[i];
            const float *f = f_h + (int64_t)h * 3 * N + 3 * i;
            welford_update(head_first + h, f[0] - fx, f_mean + 3 * c, f_m2 + 3 * c);
            welford_update(head_first + h, f[1] - fy, f_mean + 3 * c + 1, f_m2 + 3 * c + 1);
            welford_update(head_first + h, f[2] - fz, f_mean + 3 * c + 2, f_m2 + 3 * c + 2);
        }
    }
}

template <int NR, int NB>
static int pair_backward_heads_lpa(gmnn_system *s, cudaStream_t st, int lpa, int head_first, int n_heads, float *f_mean,
                                   float *f_m2) {
    const gmnn_model *m = s->model;
    if (!(s->force_mode == GMNN_FORCE_PAIRBUF && s->list_has_rev && s->rev && s->ens_gbuf && s->ens_f)) {
        set_error("batched pair backward needs the pair-buffer force mode and its batch buffers");
        return GMNN_INVALID_ARG;
    }
    const int beta_floats = (m->rp.n_species * m->rp.n_species * NR * m->rp.kb + 3) & ~3;
    const int groups = 128 / lpa;
    // heads per chunk: at most PB_HC, and at most what 96 KB of shared memory hold beside the table
    int hc = (96 * 1024 - (int)sizeof(float) * beta_floats) / (groups * NR * PSI * (int)sizeof(float));
    hc = hc > PB_HC ? PB_HC : (hc < 1 ? 1 : hc);
    hc = hc > n_heads ? n_heads : hc;
    const size_t smem = sizeof(float) * (beta_floats + (size_t)groups * hc * NR * PSI + (size_t)3 * hc * 128);
    const dim3 grid(nblocks(s->N * lpa, 128), (unsigned)((n_heads + hc - 1) / hc));
    const bool general = m->rp.basis_kind != 0 || m->rp.zbl_on;
#define GMNN_PBH_LAUNCH(L, GEN)                                                                                      \
    k_pair_backward_heads<NR, NB, L, GEN><<<grid, 128, smem, st>>>(s->N, s->pos4, s->nbr, s->count, s->cap, s->geo, m->rp, \
                                                                  m->beta, s->ens_A, s->ens_f, s->rev, s->ens_gbuf, n_heads, hc)
#define GMNN_PBH(L)                                                                                                  \
    case L: {                                                                                                        \
        static size_t opted_on[MAX_DEVICES] = {};                                                                    \
        size_t &opted = opted_on[current_device()];                                                                  \
        if (smem > 48 * 1024 && smem > opted) {                                                                      \
            GMNN_CUDA(cudaFuncSetAttribute(k_pair_backward_heads<NR, NB, L, false>,                                  \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                 \
            GMNN_CUDA(cudaFuncSetAttribute(k_pair_backward_heads<NR, NB, L, true>,                                   \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                 \
            opted = smem;                                                                                            \
        }                                                                                                            \
        if (general) GMNN_PBH_LAUNCH(L, true);                                                                       \
        else GMNN_PBH_LAUNCH(L, false);                                                                              \
    } break;
    switch (lpa) {
        GMNN_PBH(1) GMNN_PBH(2) GMNN_PBH(4) GMNN_PBH(8) GMNN_PBH(16) GMNN_PBH(32)
        default:
            set_error("lanes_per_atom must be 1, 2, 4, 8, 16 or 32");
            return GMNN_INVALID_ARG;
    }
#undef GMNN_PBH
#undef GMNN_PBH_LAUNCH
    GMNN_LAUNCHED();
    k_force_reduce_heads<8><<<nblocks(s->N * 8, 256), 256, 0, st>>>(s->N, s->count, s->cap, s->ens_gbuf, s->ens_f, s->perm,
                                                                   head_first, n_heads, f_mean, f_m2);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

// a12, batched: pair backward and force statistics of heads [head_first, head_first + n_heads) of the ensemble, whose
// adjoints are the batch in ens_A (n_heads = s->ens_batch)
int launch_pair_backward_heads_welford(gmnn_system *s, int head_first, int n_heads, float *f_mean, float *f_m2, cudaStream_t st) {
    const gmnn_model *m = s->model;
    if (m->hp.n_radial == 5 && m->hp.n_basis == 7)
        return pair_backward_heads_lpa<5, 7>(s, st, pick_lpa(s, true), head_first, n_heads, f_mean, f_m2);
    set_error("pair kernels are instantiated for n_radial = 5, n_basis = 7 only");
    return GMNN_UNSUPPORTED;
}

// wf_head >= 0: the ensemble pass of head wf_head; the force goes into the Welford statistics (f_mean, f_m2: caller order)
template <int NR, int NB>
static int pair_backward_lpa(gmnn_system *s, cudaStream_t st, int lpa, int wf_head = -1, float *f_mean = nullptr,
                             float *f_m2 = nullptr) {
    const gmnn_model *m = s->model;
    const int beta_floats = (m->rp.n_species * m->rp.n_species * NR * m->rp.kb + 3) & ~3;
    const size_t smem = sizeof(float) * (beta_floats + (128 / lpa) * NR * PSI);
    const unsigned grid = nblocks(s->N * lpa, 128);
    const bool pairbuf = s->force_mode == GMNN_FORCE_PAIRBUF;
    const int a_heads = s->ens_batch > 1 ? s->ens_batch : 1;  // batched ensemble pass: adjoints of head s->ens_head
    const bool virial = s->want_virial && s->vir_atom != nullptr;
    const bool general = virial || m->rp.basis_kind != 0 || m->rp.zbl_on;
    if (pairbuf && !(s->list_has_rev && s->rev && s->gbuf)) {
        set_error("force_mode changed after the list was built: call gmnn_build_neighbors again");
        return GMNN_INVALID_ARG;
    }
#define GMNN_PB_LAUNCH(L, PB, GEN)                                                                         \
    k_pair_backward<NR, NB, L, PB, GEN><<<grid, 128, smem, st>>>(s->N, s->pos4, s->nbr, s->count, s->cap, s->geo, m->rp, \
                                                                m->beta, a_heads > 1 ? s->ens_A : s->A, s->f_int, PB ? s->rev : nullptr, \
                                                                PB ? s->gbuf : nullptr, s->mrow, (GEN && virial) ? s->vir_atom : nullptr, \
                                                                a_heads, s->ens_head)
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
        if (pairbuf && general) GMNN_PB_LAUNCH(L, true, true);                                             \
        else if (pairbuf) GMNN_PB_LAUNCH(L, true, false);                                                  \
        else if (general) GMNN_PB_LAUNCH(L, false, true);                                                  \
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
        if (wf_head >= 0)
            k_force_reduce<8, true><<<nblocks(s->N * 8, 256), 256, 0, st>>>(s->N, s->count, s->cap, s->gbuf, s->f_int, s->perm,
                                                                           wf_head, f_mean, f_m2);
        else
            k_force_reduce<8, false><<<nblocks(s->N * 8, 256), 256, 0, st>>>(s->N, s->count, s->cap, s->gbuf, s->f_int, nullptr, 0,
                                                                            nullptr, nullptr);
        GMNN_LAUNCHED();
    } else if (wf_head >= 0) {
        k_welford_perm<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, s->f_int, s->perm, wf_head, f_mean, f_m2);
        GMNN_LAUNCHED();
    }
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_pair_backward(gmnn_system *s, cudaStream_t st) {
    const gmnn_model *m = s->model;
    if (m->hp.n_radial == 5 && m->hp.n_basis == 7) return pair_backward_lpa<5, 7>(s, st, pick_lpa(s, true));
    set_error("pair kernels are instantiated for n_radial = 5, n_basis = 7 only");
    return GMNN_UNSUPPORTED;
}

// a12: pair backward of one head of the shallow ensemble, its force folded into the running statistics over the heads
int launch_pair_backward_welford(gmnn_system *s, int head, float *f_mean, float *f_m2, cudaStream_t st) {
    const gmnn_model *m = s->model;
    if (m->hp.n_radial == 5 && m->hp.n_basis == 7) return pair_backward_lpa<5, 7>(s, st, pick_lpa(s, true), head, f_mean, f_m2);
    set_error("pair kernels are instantiated for n_radial = 5, n_basis = 7 only");
    return GMNN_UNSUPPORTED;
}

}  // namespace gmnn
