// pair_common.cuh -- what the two pair kernels share (pair_forward.cu, pair_backward.cu): the geometry of one
// packed neighbour entry, the radial basis with the cosine cutoff, the 20 unique monomials of a unit vector,
// and the lanes-per-atom choice.  (PAPER.md:49-52.)
#pragma once

#include "gmnn_internal.h"

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
// GENERAL = false: the instantiation for the configs' model (Gaussians, no ZBL); GENERAL = true adds the run-time
// switches of the other basis (and, in the kernels, the ZBL term and the virial) -- kept out of the default path,
// where the extra branches and live values cost 40 % on k_pair_forward.
template <int NB, bool WITH_DERIV, bool GENERAL>
__device__ __forceinline__ void radial_basis(const RadialParams &rp, float r, float rinv, float *phi, float *dphi,
                                             float &fc, float &dfc) {
    const float t = r * rp.inv_rc;
    if (GENERAL && rp.basis_kind == 1) {
        // Bessel-like functions of Kocer et al. (reading R30): f_n = c_n [sinc(a_{n+1} r) + sinc(a_{n+2} r)],
        // a_k = k pi / r_cut.  sin and cos of k pi t, k = 1 .. NB + 1, by the Chebyshev recurrence from the sine and
        // cosine of pi t that the cutoff function needs anyway; d/dr sinc(a r) = (cos(a r) - sinc(a r)) / r.
        float sn, cs;
        sincospif(t, &sn, &cs);
        fc = 0.5f + 0.5f * cs;
        dfc = -0.5f * PI_F * rp.inv_rc * sn;
        const float inv_pt = rinv * rp.r_cut * (1.f / PI_F);  // 1 / (pi t)
        const float two_c = 2.f * cs;
        float s_prev = 0.f, s_cur = sn, c_prev = 1.f, c_cur = cs;
        float sinc_prev = 0.f, cos_prev = 0.f;
#pragma unroll
        for (int k = 1; k <= NB + 1; ++k) {
            const float sinc_k = s_cur * inv_pt * (1.f / (float)k);
            if (k >= 2) {
                phi[k - 2] = rp.bessel_c[k - 2] * (sinc_prev + sinc_k);
                if (WITH_DERIV) dphi[k - 2] = rp.bessel_c[k - 2] * ((cos_prev - sinc_prev) + (c_cur - sinc_k)) * rinv;
            }
            sinc_prev = sinc_k, cos_prev = c_cur;
            const float s_next = fmaf(two_c, s_cur, -s_prev), c_next = fmaf(two_c, c_cur, -c_prev);
            s_prev = s_cur, s_cur = s_next, c_prev = c_cur, c_cur = c_next;
        }
        return;
    }
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

// ZBL repulsion (reading R31) of one directed pair: e = V / 2 and, WITH_DERIV, de = d(V/2)/dr;
// V = scale k_e Z1 Z2 / r phi(r / a) 1/2 [1 + cos(pi r / r_max)], a = 0.8854 a_0 / (Z1^0.23 + Z2^0.23).  r2 < zbl_r_max2.
template <bool WITH_DERIV>
__device__ __forceinline__ void zbl_half(const RadialParams &rp, int zi, int zj, float r, float rinv, float &e, float &de) {
    const float inv_a = (rp.zbl_zpow[zi] + rp.zbl_zpow[zj]) * (1.f / (0.8854f * 0.529177f));
    const float x = r * inv_a;
    const float e0 = 0.1818f * __expf(-3.2f * x), e1 = 0.5099f * __expf(-0.9423f * x), e2 = 0.2802f * __expf(-0.4029f * x),
                e3 = 0.02817f * __expf(-0.2016f * x);
    const float phi = (e0 + e1) + (e2 + e3);
    const float coul = rp.zbl_pref * rp.zbl_z[zi] * rp.zbl_z[zj] * rinv;
    float sn, cs;
    sincospif(r * rp.zbl_inv_rmax, &sn, &cs);
    const float fcz = 0.5f + 0.5f * cs;
    e = coul * phi * fcz;
    if (WITH_DERIV) {
        const float dphi = -inv_a * ((3.2f * e0 + 0.9423f * e1) + (0.4029f * e2 + 0.2016f * e3));
        const float dfcz = -0.5f * PI_F * rp.zbl_inv_rmax * sn;
        de = coul * (fcz * (dphi - phi * rinv) + phi * dfcz);
    }
}

__device__ __forceinline__ void monomials(float x, float y, float z, float *m) {
    m[0] = 1.f;
    m[1] = x; m[2] = y; m[3] = z;
    m[4] = x * x; m[5] = x * y; m[6] = x * z; m[7] = y * y; m[8] = y * z; m[9] = z * z;
    m[10] = m[4] * x; m[11] = m[4] * y; m[12] = m[4] * z; m[13] = m[7] * x; m[14] = m[5] * z;
    m[15] = m[9] * x; m[16] = m[7] * y; m[17] = m[7] * z; m[18] = m[9] * y; m[19] = m[9] * z;
}


static inline unsigned nblocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }

static int pick_lpa(const gmnn_system *s, bool backward = false) {
    if (s->lanes_per_atom > 0) return s->lanes_per_atom;
    // enough warps to fill 148 SMs several times over: small systems spread one atom over more lanes.  Measured at config 5
    // (1 048 576 atoms, round 2): k_pair_forward 1.44 / 1.58 / 1.99 ms at 2 / 4 / 8 lanes, k_pair_backward + k_force_reduce
    // 4.55 / 3.33 / 2.99 / 3.17 ms at 1 / 2 / 4 / 8 (its A_i staging in shared memory is shared by the lanes of an atom)
    if (s->N >= 262144) return backward ? 4 : 2;
    if (s->N >= 65536) return 4;
    if (s->N >= 8192) return 8;
    return 32;
}

}  // namespace gmnn
