// contraction.cuh -- invariants G_i from the moments Psi_i and the adjoint of that map, in
// symmetry-unique storage (Eq. 3; DESIGN.md section 3 readings R7, R8).
//
// A channel s of an atom holds 20 numbers, the sums over neighbours of R_s times the unique
// monomials of the unit bond vector u = (x, y, z):
//   m  0      : 1                                   (L = 0)
//   m  1.. 3  : x y z                               (L = 1)
//   m  4.. 9  : xx xy xz yy yz zz                   (L = 2), multiplicity 1 2 2 1 2 1
//   m 10..19  : xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz (L = 3), multiplicity 1 3 3 3 6 3 1 3 3 1
// A full contraction over Cartesian indices becomes a sum over unique components weighted by the
// multiplicity.  Blocks and their order (lexicographic in the channel tuple):
//   0: P0[s]   1: P1.P1 (s1<=s2)   2: P2:P2 (s1<=s2)   3: P3:.P3 (s1<=s2)
//   4: tr(P2 P2 P2) (s1<=s2<=s3)   5: P1 P2 P1 (s1<=s2, s3)   6: P3 P3 P2 (s1<=s2, s3)
//   7: P1 P3 P2 (s1, s2, s3)
// Every loop below has compile-time bounds and is fully unrolled, so with register-resident
// accessors the result is straight-line FMA code with constant indices.
//
// contract_backward is the reverse mode of contract_forward, statement by statement: the
// adjoint A[s][m] = dE/dPsi[s][m] with respect to the UNIQUE variables, which is exactly the
// coefficient of monomial m in the per-pair polynomial used by the pair backward kernel.
#pragma once

#if defined(__CUDACC__)
#define GMNN_HD __host__ __device__ __forceinline__
#else
#define GMNN_HD inline
#endif

namespace gmnn {

constexpr int NM = 20;  // unique monomials per channel
constexpr int M1 = 1, M2 = 4, M3 = 10;

GMNN_HD constexpr int idx2(int a, int b) {
    int lo = a < b ? a : b, hi = a < b ? b : a;
    return lo == 0 ? hi : (lo == 1 ? 2 + hi : 5);
}
GMNN_HD constexpr int idx3(int a, int b, int c) {
    // sort the triple, then rank among 000 001 002 011 012 022 111 112 122 222
    int lo = a < b ? (a < c ? a : c) : (b < c ? b : c);
    int hi = a > b ? (a > c ? a : c) : (b > c ? b : c);
    int mid = a + b + c - lo - hi;
    return lo == 0 ? (mid == 0 ? hi : (mid == 1 ? 2 + hi : 5)) : (lo == 1 ? (mid == 1 ? 5 + hi : 8) : 9);
}
GMNN_HD constexpr float mult2(int u) { return (u == 0 || u == 3 || u == 5) ? 1.f : 2.f; }
GMNN_HD constexpr float mult3(int u) { return (u == 0 || u == 6 || u == 9) ? 1.f : (u == 4 ? 6.f : 3.f); }
// first/second Cartesian index of unique pair u2
GMNN_HD constexpr int u2a(int u) { return u < 3 ? 0 : (u < 5 ? 1 : 2); }
GMNN_HD constexpr int u2b(int u) { return u < 3 ? u : (u < 5 ? u - 2 : 2); }

template <int NR>
struct Feat {
    static constexpr int NP = NR * (NR + 1) / 2;
    static constexpr int NT = NR * (NR + 1) * (NR + 2) / 6;
    static constexpr int OFF0 = 0, OFF1 = NR, OFF2 = OFF1 + NP, OFF3 = OFF2 + NP, OFF4 = OFF3 + NP;
    static constexpr int OFF5 = OFF4 + NT, OFF6 = OFF5 + NP * NR, OFF7 = OFF6 + NP * NR;
    static constexpr int N = OFF7 + NR * NR * NR;
    GMNN_HD static constexpr int pidx(int s1, int s2) { return s1 * NR - s1 * (s1 - 1) / 2 + (s2 - s1); }
    GMNN_HD static constexpr int tidx(int s1, int s2, int s3) {
        int r = 0;
        for (int a = 0; a < s1; ++a) r += (NR - a) * (NR - a + 1) / 2;
        for (int b = s1; b < s2; ++b) r += NR - b;
        return r + (s3 - s2);
    }
};

// P(s, m) -> float;  emit(f, value) with f a compile-time constant after unrolling.
// BLOCKS: bit k set = evaluate block k (bits 0-3 share one loop nest and go together).
template <int NR, int BLOCKS = 0xFF, class PGet, class Emit>
GMNN_HD void contract_forward(PGet P, Emit emit) {
    using F = Feat<NR>;
    if constexpr ((BLOCKS & 0xF) != 0) {
#pragma unroll
    for (int s = 0; s < NR; ++s) emit(F::OFF0 + s, P(s, 0));
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            float v1 = 0.f, v2 = 0.f, v3 = 0.f;
#pragma unroll
            for (int a = 0; a < 3; ++a) v1 = fmaf(P(s1, M1 + a), P(s2, M1 + a), v1);
#pragma unroll
            for (int u = 0; u < 6; ++u) v2 = fmaf(mult2(u) * P(s1, M2 + u), P(s2, M2 + u), v2);
#pragma unroll
            for (int u = 0; u < 10; ++u) v3 = fmaf(mult3(u) * P(s1, M3 + u), P(s2, M3 + u), v3);
            emit(F::OFF1 + F::pidx(s1, s2), v1);
            emit(F::OFF2 + F::pidx(s1, s2), v2);
            emit(F::OFF3 + F::pidx(s1, s2), v3);
        }
    }
    }
    // block 4: tr(X Y Z), X = P2[s1], Y = P2[s2], Z = P2[s3]
    if constexpr ((BLOCKS & 0x10) != 0) {
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            float S[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    float m = 0.f;
#pragma unroll
                    for (int c = 0; c < 3; ++c) m = fmaf(P(s1, M2 + idx2(a, c)), P(s2, M2 + idx2(c, b)), m);
                    S[idx2(a, b)] += m;
                }
#pragma unroll
            for (int s3 = s2; s3 < NR; ++s3) {
                float v = 0.f;
#pragma unroll
                for (int u = 0; u < 6; ++u) v = fmaf(S[u], P(s3, M2 + u), v);
                emit(F::OFF4 + F::tidx(s1, s2, s3), v);
            }
        }
    }
    }
    // block 5: p_a q_b Z_ab, p = P1[s1], q = P1[s2], Z = P2[s3]
    if constexpr ((BLOCKS & 0x20) != 0) {
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            float O[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) O[idx2(a, b)] = fmaf(P(s1, M1 + a), P(s2, M1 + b), O[idx2(a, b)]);
#pragma unroll
            for (int s3 = 0; s3 < NR; ++s3) {
                float v = 0.f;
#pragma unroll
                for (int u = 0; u < 6; ++u) v = fmaf(O[u], P(s3, M2 + u), v);
                emit(F::OFF5 + F::pidx(s1, s2) * NR + s3, v);
            }
        }
    }
    }
    // block 6: X_abc Y_abd Z_cd, X = P3[s1], Y = P3[s2], Z = P2[s3]
    if constexpr ((BLOCKS & 0x40) != 0) {
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            float S[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    float n = 0.f;
#pragma unroll
                    for (int u = 0; u < 6; ++u)
                        n = fmaf(mult2(u) * P(s1, M3 + idx3(u2a(u), u2b(u), c)), P(s2, M3 + idx3(u2a(u), u2b(u), d)), n);
                    S[idx2(c, d)] += n;
                }
#pragma unroll
            for (int s3 = 0; s3 < NR; ++s3) {
                float v = 0.f;
#pragma unroll
                for (int u = 0; u < 6; ++u) v = fmaf(S[u], P(s3, M2 + u), v);
                emit(F::OFF6 + F::pidx(s1, s2) * NR + s3, v);
            }
        }
    }
    }
    // block 7: p_a X_abc Z_bc, p = P1[s1], X = P3[s2], Z = P2[s3]
    if constexpr ((BLOCKS & 0x80) != 0) {
#pragma unroll
    for (int s2 = 0; s2 < NR; ++s2) {
#pragma unroll
        for (int s3 = 0; s3 < NR; ++s3) {
            float T[3] = {0.f, 0.f, 0.f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int u = 0; u < 6; ++u)
                    T[a] = fmaf(mult2(u) * P(s2, M3 + idx3(a, u2a(u), u2b(u))), P(s3, M2 + u), T[a]);
#pragma unroll
            for (int s1 = 0; s1 < NR; ++s1) {
                float v = 0.f;
#pragma unroll
                for (int a = 0; a < 3; ++a) v = fmaf(P(s1, M1 + a), T[a], v);
                emit(F::OFF7 + (s1 * NR + s2) * NR + s3, v);
            }
        }
    }
    }
}

// P(s, m) -> float;  g(f) -> float (dE/dG_f);  acc(s, m, value): A[s][m] += value.
struct NoStep {
    GMNN_HD void operator()() const {}
};

// step(): called after every channel-pair iteration of the straight-line body (a kernel can put a block
// barrier there to keep its warps inside the same stretch of code).
//
// ORBIT = true evaluates only one representative of every orbit of channel tuples under the cyclic shift
// s -> s + 1 (mod NR) of ALL channels: pairs {0, 0}, {0, 1}, ... {0, NR/2}; block 4 multisets {0,0,s3},
// {0,1,2}, {0,1,3}; block 7 tuples with s2 = 0.  Every block is symmetric under the exchanges its loops
// skip (s1 <-> s2; any permutation in block 4), so a caller that runs the representatives NR times, each
// time with P and the adjoints renumbered s -> s + 1 and g looked up at the shifted tuple, covers every
// tuple exactly once with a fifth of the code (k_contract_backward, descriptor.cu).  NR must be prime.
template <int NR>
GMNN_HD constexpr bool orbit_pair(int s1, int s2) { return s1 == 0 && s2 <= NR / 2; }
template <int NR>
GMNN_HD constexpr bool orbit_triple(int s1, int s2, int s3) {
    return s1 == 0 && (s2 == 0 || (s2 == 1 && (s3 == 2 || s3 == 3)));
}

template <int NR, int BLOCKS = 0xFF, bool ORBIT = false, class PGet, class GGet, class Acc, class Step = NoStep>
GMNN_HD void contract_backward(PGet P, GGet g, Acc acc, Step step = Step()) {
    using F = Feat<NR>;
    static_assert(!ORBIT || NR == 5, "orbit representatives are written out for NR = 5");
    if constexpr ((BLOCKS & 0xF) != 0) {
#pragma unroll
    for (int s = 0; s < (ORBIT ? 1 : NR); ++s) acc(s, 0, g(F::OFF0 + s));
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            if (ORBIT && !orbit_pair<NR>(s1, s2)) continue;
            step();
            const float g1 = g(F::OFF1 + F::pidx(s1, s2));
            const float g2 = g(F::OFF2 + F::pidx(s1, s2));
            const float g3 = g(F::OFF3 + F::pidx(s1, s2));
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                acc(s1, M1 + a, g1 * P(s2, M1 + a));
                acc(s2, M1 + a, g1 * P(s1, M1 + a));
            }
#pragma unroll
            for (int u = 0; u < 6; ++u) {
                acc(s1, M2 + u, g2 * mult2(u) * P(s2, M2 + u));
                acc(s2, M2 + u, g2 * mult2(u) * P(s1, M2 + u));
            }
#pragma unroll
            for (int u = 0; u < 10; ++u) {
                acc(s1, M3 + u, g3 * mult3(u) * P(s2, M3 + u));
                acc(s2, M3 + u, g3 * mult3(u) * P(s1, M3 + u));
            }
        }
    }
    }
    // block 4
    if constexpr ((BLOCKS & 0x10) != 0) {
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            if (ORBIT && !orbit_triple<NR>(s1, s2, s2 == 0 ? 0 : 2)) continue;  // pairs (0,0) and (0,1)
            step();
            float S[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    float m = 0.f;
#pragma unroll
                    for (int c = 0; c < 3; ++c) m = fmaf(P(s1, M2 + idx2(a, c)), P(s2, M2 + idx2(c, b)), m);
                    S[idx2(a, b)] += m;
                }
            float dS[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int s3 = s2; s3 < NR; ++s3) {
                if (ORBIT && !orbit_triple<NR>(s1, s2, s3)) continue;
                const float gv = g(F::OFF4 + F::tidx(s1, s2, s3));
#pragma unroll
                for (int u = 0; u < 6; ++u) {
                    dS[u] = fmaf(gv, P(s3, M2 + u), dS[u]);
                    acc(s3, M2 + u, gv * S[u]);
                }
            }
            // M = X Y, dM_ab = dS[idx2(a,b)] =: D (symmetric).  dX = D Y, dY = X D (X, Y symmetric).
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    float dx = 0.f, dy = 0.f;
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        dx = fmaf(dS[idx2(a, b)], P(s2, M2 + idx2(b, c)), dx);  // (D Y)_ac
                        dy = fmaf(P(s1, M2 + idx2(a, b)), dS[idx2(b, c)], dy);  // (X D)_ac
                    }
                    acc(s1, M2 + idx2(a, c), dx);
                    acc(s2, M2 + idx2(a, c), dy);
                }
        }
    }
    }
    // block 5
    if constexpr ((BLOCKS & 0x20) != 0) {
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            if (ORBIT && !orbit_pair<NR>(s1, s2)) continue;
            step();
            float O[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) O[idx2(a, b)] = fmaf(P(s1, M1 + a), P(s2, M1 + b), O[idx2(a, b)]);
            float dO[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int s3 = 0; s3 < NR; ++s3) {
                const float gv = g(F::OFF5 + F::pidx(s1, s2) * NR + s3);
#pragma unroll
                for (int u = 0; u < 6; ++u) {
                    dO[u] = fmaf(gv, P(s3, M2 + u), dO[u]);
                    acc(s3, M2 + u, gv * O[u]);
                }
            }
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                float dp = 0.f, dq = 0.f;
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    dp = fmaf(dO[idx2(a, b)], P(s2, M1 + b), dp);
                    dq = fmaf(dO[idx2(b, a)], P(s1, M1 + b), dq);
                }
                acc(s1, M1 + a, dp);
                acc(s2, M1 + a, dq);
            }
        }
    }
    }
    // block 6
    if constexpr ((BLOCKS & 0x40) != 0) {
#pragma unroll
    for (int s1 = 0; s1 < NR; ++s1) {
#pragma unroll
        for (int s2 = s1; s2 < NR; ++s2) {
            if (ORBIT && !orbit_pair<NR>(s1, s2)) continue;
            step();
            float S[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    float n = 0.f;
#pragma unroll
                    for (int u = 0; u < 6; ++u)
                        n = fmaf(mult2(u) * P(s1, M3 + idx3(u2a(u), u2b(u), c)), P(s2, M3 + idx3(u2a(u), u2b(u), d)), n);
                    S[idx2(c, d)] += n;
                }
            float dS[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int s3 = 0; s3 < NR; ++s3) {
                const float gv = g(F::OFF6 + F::pidx(s1, s2) * NR + s3);
#pragma unroll
                for (int u = 0; u < 6; ++u) {
                    dS[u] = fmaf(gv, P(s3, M2 + u), dS[u]);
                    acc(s3, M2 + u, gv * S[u]);
                }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const float dn = dS[idx2(c, d)];
#pragma unroll
                    for (int u = 0; u < 6; ++u) {
                        acc(s1, M3 + idx3(u2a(u), u2b(u), c), mult2(u) * dn * P(s2, M3 + idx3(u2a(u), u2b(u), d)));
                        acc(s2, M3 + idx3(u2a(u), u2b(u), d), mult2(u) * dn * P(s1, M3 + idx3(u2a(u), u2b(u), c)));
                    }
                }
        }
    }
    }
    // block 7
    if constexpr ((BLOCKS & 0x80) != 0) {
#pragma unroll
    for (int s2 = 0; s2 < (ORBIT ? 1 : NR); ++s2) {
#pragma unroll
        for (int s3 = 0; s3 < NR; ++s3) {
            step();
            float T[3] = {0.f, 0.f, 0.f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int u = 0; u < 6; ++u)
                    T[a] = fmaf(mult2(u) * P(s2, M3 + idx3(a, u2a(u), u2b(u))), P(s3, M2 + u), T[a]);
            float dT[3] = {0.f, 0.f, 0.f};
#pragma unroll
            for (int s1 = 0; s1 < NR; ++s1) {
                const float gv = g(F::OFF7 + (s1 * NR + s2) * NR + s3);
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    dT[a] = fmaf(gv, P(s1, M1 + a), dT[a]);
                    acc(s1, M1 + a, gv * T[a]);
                }
            }
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int u = 0; u < 6; ++u) {
                    acc(s2, M3 + idx3(a, u2a(u), u2b(u)), mult2(u) * dT[a] * P(s3, M2 + u));
                    acc(s3, M2 + u, mult2(u) * dT[a] * P(s2, M3 + idx3(a, u2a(u), u2b(u))));
                }
        }
    }
    }
}

}  // namespace gmnn
