// neighbor.cu -- cell binning, deterministic cell sort and Verlet-list build (SURVEY.md 8(a) rows
// a1-a3; PAPER.md:169-171 neighbour list with skin, :171 several images in small cells, :381).
//
// Data layout.  Atoms are renumbered into cell order ("internal" order, perm[k] = caller index of
// internal atom k; inside a cell atoms are ordered by caller index, so the order is a pure
// function of the positions).  pos4[k] = (x, y, z, species bits): one 16-byte gather per
// neighbour in every later kernel.  The list is row-major nbr[k][cap] of packed entries
//   entry = j | (nx+4) << 22 | (ny+4) << 25 | (nz+4) << 28,   j internal, n the image vector,
// so a group of lanes reads a contiguous run of one atom's row with 16-byte loads.
//
// Membership predicate (reading R20), unfused fp32, identical to the oracle's:
//   s_a = fl(n_a L_a); d_a = fl(fl(x_j,a - x_i,a) + s_a); r2 = fl(fl(dx dx + dy dy) + dz dz) < fl(r_list^2)
//
// Every kernel of the rebuild takes (cond, thr2): inside gmnn_md_verlet_steps the rebuild is
// launched every step and exits immediately unless the squared max displacement stored in *cond
// exceeds thr2 -- the loop never synchronises with the host.
#include "gmnn_internal.h"

namespace gmnn {

__device__ __forceinline__ bool skip_rebuild(const int32_t *cond, float thr2) {
    return cond != nullptr && __int_as_float(*((const volatile int32_t *)cond)) <= thr2;
}

// fractional coordinate a of position p in a general lattice
__device__ __forceinline__ float frac_coord(const Geometry &g, const float *p, int a) {
    return p[0] * g.hinv[a] + p[1] * g.hinv[3 + a] + p[2] * g.hinv[6 + a];
}

__global__ void k_wrap(int64_t N, float *x, Geometry g, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    if (g.triclinic) {  // fold in fractional coordinates: x -= floor(s_a) a_a on the periodic axes
        for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < N; i += gridDim.x * (int64_t)blockDim.x) {
            float p[3] = {x[3 * i], x[3 * i + 1], x[3 * i + 2]};
            for (int pass = 0; pass < 2; ++pass)  // the second pass catches a rounding step across a face
                for (int a = 0; a < 3; ++a) {
                    if (!g.pbc[a]) continue;
                    const float k = floorf(frac_coord(g, p, a));
                    if (k != 0.f) {
                        p[0] -= k * g.h[3 * a], p[1] -= k * g.h[3 * a + 1], p[2] -= k * g.h[3 * a + 2];
                    }
                }
            x[3 * i] = p[0], x[3 * i + 1] = p[1], x[3 * i + 2] = p[2];
        }
        return;
    }
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < 3 * N; t += gridDim.x * (int64_t)blockDim.x) {
        int a = (int)(t % 3);
        if (!g.pbc[a]) continue;
        float v = x[t];
        v -= g.L[a] * floorf(v * g.invL[a]);
        if (!(v >= 0.f) || v >= g.L[a]) v = 0.f;
        x[t] = v;
    }
}

__global__ void k_zero_cells(int64_t ncells, int32_t *cell_count, int32_t *cell_fill, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t <= ncells; t += gridDim.x * (int64_t)blockDim.x) {
        cell_count[t] = 0;
        if (t < ncells) cell_fill[t] = 0;
    }
}

__device__ __forceinline__ int cell_coord(float x, float inv_edge, int nc) {
    int c = (int)floorf(x * inv_edge);
    return c < 0 ? 0 : (c >= nc ? nc - 1 : c);
}
// cell index along axis a of position p: slabs in x for diag(L), in fractional coordinates for a general lattice
__device__ __forceinline__ int cell_coord_of(const Geometry &g, const float *p, int a) {
    if (!g.triclinic) return cell_coord(p[a], g.inv_edge[a], g.ncell[a]);
    return cell_coord(frac_coord(g, p, a), (float)g.ncell[a], g.ncell[a]);
}

__global__ void k_cell_assign(int64_t N, const float *__restrict__ x, Geometry g, int32_t *cell_of,
                              int32_t *cell_count, int32_t *flags, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < N; i += gridDim.x * (int64_t)blockDim.x) {
        float p[3] = {x[3 * i], x[3 * i + 1], x[3 * i + 2]};
        int c[3];
        bool bad = false;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (g.triclinic) {  // inside the cell up to the rounding of the fractional coordinate
                const float f = frac_coord(g, p, a);
                bad |= !(f >= -1e-5f && f < 1.f + 1e-5f);
            } else {
                bad |= !(p[a] >= 0.f && p[a] < g.L[a]);
            }
            c[a] = cell_coord_of(g, p, a);
        }
        if (bad) flags[FLAG_OUT_OF_BOX] = 1;
        int cid = (c[2] * g.ncell[1] + c[1]) * g.ncell[0] + c[0];
        cell_of[i] = cid;
        atomicAdd(&cell_count[cid], 1);
    }
}

// Exclusive scan of cell_count[0..n) into cell_start[0..n]; one block of 1024 threads.
__global__ void k_scan_cells(int64_t n, const int32_t *__restrict__ cnt, int32_t *start, const int32_t *cond,
                             float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    __shared__ int32_t warp_sums[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int64_t per = (n + blockDim.x - 1) / blockDim.x;
    const int64_t b = tid * per, e = (b + per < n) ? b + per : n;
    int32_t local = 0;
    for (int64_t q = b; q < e; ++q) local += cnt[q];
    int32_t incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int32_t w = warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int32_t v = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += v;
        }
        warp_sums[lane] = w;
    }
    __syncthreads();
    int32_t run = incl - local + (wid > 0 ? warp_sums[wid - 1] : 0);
    for (int64_t q = b; q < e; ++q) {
        start[q] = run;
        run += cnt[q];
    }
    if (tid == blockDim.x - 1) start[n] = warp_sums[31];
}

__global__ void k_cell_fill(int64_t N, const int32_t *__restrict__ cell_of, const int32_t *__restrict__ cell_start,
                            int32_t *cell_fill, int32_t *slot_tmp, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < N; i += gridDim.x * (int64_t)blockDim.x) {
        int c = cell_of[i];
        int slot = atomicAdd(&cell_fill[c], 1);
        slot_tmp[cell_start[c] + slot] = (int32_t)i;
    }
}

// The atomics above fill a cell in arbitrary order; rank every atom inside its cell by caller
// index so that the internal numbering (and with it every summation order) is reproducible.
__global__ void k_cell_rank(int64_t N, const int32_t *__restrict__ slot_tmp, const int32_t *__restrict__ cell_of,
                            const int32_t *__restrict__ cell_start, int32_t *perm, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < N; k += gridDim.x * (int64_t)blockDim.x) {
        int i = slot_tmp[k];
        int c = cell_of[i];
        int b = cell_start[c], e = cell_start[c + 1];
        int rank = 0;
        for (int q = b; q < e; ++q) rank += (slot_tmp[q] < i);
        perm[b + rank] = i;
    }
}

// pos4 (internal order) from the caller's positions; at a build also the reference copy xref;
// otherwise the skin test of gmnn_energy_forces (GMNN_STALE_NEIGHBORS).
__global__ void k_gather(int64_t N, const float *__restrict__ x, const int32_t *__restrict__ species,
                         const int32_t *__restrict__ perm, float4 *pos4, float *xref, bool is_build,
                         float half_skin2, int32_t *flags, const int32_t *cond, float thr2) {
    if (is_build && skip_rebuild(cond, thr2)) return;
    int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= N) return;
    int i = perm[k];
    float px = x[3 * (int64_t)i], py = x[3 * (int64_t)i + 1], pz = x[3 * (int64_t)i + 2];
    pos4[k] = make_float4(px, py, pz, __int_as_float(species[i]));
    if (is_build) {
        xref[3 * (int64_t)i] = px;
        xref[3 * (int64_t)i + 1] = py;
        xref[3 * (int64_t)i + 2] = pz;
    } else if (flags != nullptr) {
        float dx = px - xref[3 * (int64_t)i], dy = py - xref[3 * (int64_t)i + 1], dz = pz - xref[3 * (int64_t)i + 2];
        if (dx * dx + dy * dy + dz * dz > half_skin2) flags[FLAG_STALE] = 1;
    }
}

// squared distance in the unfused fp32 arithmetic that defines list membership (reading R20); exactly
// symmetric under i <-> j with the opposite image
__device__ __forceinline__ float list_r2(const float4 &xi, const float4 &xj, float sx, float sy, float sz) {
    float dx = __fadd_rn(__fsub_rn(xj.x, xi.x), sx);
    float dy = __fadd_rn(__fsub_rn(xj.y, xi.y), sy);
    float dz = __fadd_rn(__fsub_rn(xj.z, xi.z), sz);
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}
__device__ __forceinline__ bool in_list(const float4 &xi, const float4 &xj, float sx, float sy, float sz, float rl2) {
    return list_r2(xi, xj, sx, sy, sz) < rl2;
}

// lattice shift of the membership predicate, component x, in the unfused order reading R20 / O-16 fixes:
// fl(fl(fl(n1 a_x) + fl(n2 b_x)) + fl(n3 c_x)); with zero off-diagonals this is fl(n_x L_x) exactly
__device__ __forceinline__ float list_shift(const Geometry &g, int x, int n1, int n2, int n3) {
    return __fadd_rn(__fadd_rn(__fmul_rn((float)n1, g.h[x]), __fmul_rn((float)n2, g.h[3 + x])), __fmul_rn((float)n3, g.h[6 + x]));
}

__device__ __forceinline__ uint32_t image_code(int nx, int ny, int nz) {
    return ((uint32_t)(nx + 4) << NBR_J_BITS) | ((uint32_t)(ny + 4) << (NBR_J_BITS + 3)) |
           ((uint32_t)(nz + 4) << (NBR_J_BITS + 6));
}

constexpr int RUNS_PITCH = 56;  // 2 parts x 27 run starts, the row length at [54]

constexpr int SHELL_BUF = 256;  // skin-shell entries of one row staged in shared memory during the scan

// One warp per centre atom; lanes test 32 candidates of a neighbouring cell at a time and append
// the hits in candidate order (ballot + prefix popcount): the list order is deterministic.
// A row has two parts: first the pairs inside r_cut at build time, then the skin shell.  The pair
// kernels walk a row front to back, so the lanes of a warp reach the (mostly skipped) shell entries
// together instead of diverging entry by entry.  Inside a part, 27 cells in the fixed order
// idx = (oz+1)*9 + (oy+1)*3 + (ox+1); runs[part*27 + idx] = first slot of the cell's run (entries of
// a run ascend in atom index).  The reverse-pair index uses the runs: the partner of an entry in run
// (part, idx) sits in run (part, 26 - idx) of the partner's row (r2 is bitwise symmetric, so both
// directions fall in the same part).  One scan: inside entries go straight to the row, shell entries
// wait in shared memory until the inside count is known (rows with more than SHELL_BUF shell entries
// scan a second time).
__global__ void __launch_bounds__(256)
k_build_cells(int64_t N, const float4 *__restrict__ pos4, const int32_t *__restrict__ cell_start, Geometry g,
              uint32_t *nbr, int32_t *count, int cap, int32_t *flags, const int32_t *cond, float thr2,
              uint16_t *runs) {
    if (skip_rebuild(cond, thr2)) return;
    __shared__ uint32_t s_shell[8][SHELL_BUF];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned below = (1u << lane) - 1u;
    // grid-stride over atoms (one warp each): the launch is a few waves of blocks, so that the
    // every-step launches that skip_rebuild() turns into no-ops stay cheap
    const int64_t n_warps = (gridDim.x * (int64_t)blockDim.x) >> 5;
    for (int64_t i = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5; i < N; i += n_warps) {
        const float4 xi = pos4[i];
        const float pi3[3] = {xi.x, xi.y, xi.z};
        const int cx = cell_coord_of(g, pi3, 0), cy = cell_coord_of(g, pi3, 1), cz = cell_coord_of(g, pi3, 2);
        uint32_t *row = nbr + i * (int64_t)cap;
        // The 27 neighbouring cells are described once, lane l < 27 computing cell l (periodic wrap, candidate range in
        // the cell-sorted order, lattice shift and image code of the cell's image); the scan below takes cell idx's
        // description from lane idx by shuffles.  (Every lane recomputing every cell's description cost two thirds
        // of this kernel's 5.9 G warp instructions at config 5: it is instruction-bound.)
        int cb = 0, ce = 0;
        float csx = 0.f, csy = 0.f, csz = 0.f;
        uint32_t ccode = 0u;
        if (lane < 27) {
            const int oz = lane / 9 - 1, oy = (lane / 3) % 3 - 1, ox = lane % 3 - 1;
            bool ok = true;
            int z = cz + oz, nz = 0;
            if (z < 0) { ok = ok && g.pbc[2]; z += g.ncell[2]; nz = -1; }
            else if (z >= g.ncell[2]) { ok = ok && g.pbc[2]; z -= g.ncell[2]; nz = 1; }
            int y = cy + oy, ny = 0;
            if (y < 0) { ok = ok && g.pbc[1]; y += g.ncell[1]; ny = -1; }
            else if (y >= g.ncell[1]) { ok = ok && g.pbc[1]; y -= g.ncell[1]; ny = 1; }
            int x = cx + ox, nx = 0;
            if (x < 0) { ok = ok && g.pbc[0]; x += g.ncell[0]; nx = -1; }
            else if (x >= g.ncell[0]) { ok = ok && g.pbc[0]; x -= g.ncell[0]; nx = 1; }
            if (ok) {
                const int c = (z * g.ncell[1] + y) * g.ncell[0] + x;
                cb = cell_start[c], ce = cell_start[c + 1];
            }
            csx = list_shift(g, 0, nx, ny, nz), csy = list_shift(g, 1, nx, ny, nz), csz = list_shift(g, 2, nx, ny, nz);
            ccode = image_code(nx, ny, nz);
        }
        const uint32_t home_code = image_code(0, 0, 0);
        // visit(idx, fn): candidates of cell idx in chunks of 32; fn(entry, r2, valid) per lane
        auto visit = [&](int idx, auto fn) {
            const int b = __shfl_sync(0xffffffffu, cb, idx), e = __shfl_sync(0xffffffffu, ce, idx);
            const float sx = __shfl_sync(0xffffffffu, csx, idx), sy = __shfl_sync(0xffffffffu, csy, idx),
                        sz = __shfl_sync(0xffffffffu, csz, idx);
            const uint32_t code = __shfl_sync(0xffffffffu, ccode, idx);
            const bool home = code == home_code;
            for (int base = b; base < e; base += 32) {
                const int j = base + lane;
                const bool valid = j < e && !(home && j == (int)i);
                const float r2 = valid ? list_r2(xi, pos4[j], sx, sy, sz) : 3.0e38f;
                fn((uint32_t)j | code, r2, valid);
            }
        };
        int n_in = 0, n_out = 0;
        int run_in = 0, run_out = 0;  // lane idx: the counts when the scan reached cell idx
        for (int idx = 0; idx < 27; ++idx) {
            if (lane == idx) run_in = n_in, run_out = n_out;
            visit(idx, [&](uint32_t entry, float r2, bool valid) {
                const bool kin = valid && r2 < g.r_cut2 && r2 < g.r_list2;
                const bool kout = valid && !(r2 < g.r_cut2) && r2 < g.r_list2;
                const unsigned m_in = __ballot_sync(0xffffffffu, kin), m_out = __ballot_sync(0xffffffffu, kout);
                const int p = n_in + __popc(m_in & below), q = n_out + __popc(m_out & below);
                if (kin && p < cap) row[p] = entry;
                if (kout && q < SHELL_BUF) s_shell[wid][q] = entry;
                n_in += __popc(m_in);
                n_out += __popc(m_out);
            });
        }
        __syncwarp();
        if (n_out <= SHELL_BUF) {
            for (int q = lane; q < n_out; q += 32)
                if (n_in + q < cap) row[n_in + q] = s_shell[wid][q];
        } else {  // the shell did not fit: scan it again, now that its place in the row is known
            int q0 = n_in;
            for (int idx = 0; idx < 27; ++idx)
                visit(idx, [&](uint32_t entry, float r2, bool valid) {
                    const bool kout = valid && !(r2 < g.r_cut2) && r2 < g.r_list2;
                    const unsigned m_out = __ballot_sync(0xffffffffu, kout);
                    const int q = q0 + __popc(m_out & below);
                    if (kout && q < cap) row[q] = entry;
                    q0 += __popc(m_out);
                });
        }
        const int n = n_in + n_out;
        if (runs) {
            if (lane < 27) {
                runs[i * RUNS_PITCH + lane] = (uint16_t)(run_in < cap ? run_in : cap);
                runs[i * RUNS_PITCH + 27 + lane] = (uint16_t)(n_in + run_out < cap ? n_in + run_out : cap);
            }
            if (lane == 0) runs[i * RUNS_PITCH + 54] = (uint16_t)(n < cap ? n : cap);
        }
        if (lane == 0) {
            count[i] = n < cap ? n : cap;
            if (n > cap) atomicMax(&flags[FLAG_MAXCOUNT], n);
        }
        __syncwarp();  // s_shell is reused for the warp's next atom
    }
}

// Boxes with fewer than 3 cells on a periodic axis: explicit loop over all atoms and all images
// n in [-k..k]^3 (minimum image is not enough there).  O(N^2 images), N <= 16384.
__global__ void __launch_bounds__(256)
k_build_small(int64_t N, const float4 *__restrict__ pos4, Geometry g, uint32_t *nbr, int32_t *count, int cap,
              int32_t *flags, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    const int lane = threadIdx.x & 31;
    // grid-stride over atoms (one warp each): the launch is a few waves of blocks, so that the
    // every-step launches that skip_rebuild() turns into no-ops stay cheap
    const int64_t n_warps = (gridDim.x * (int64_t)blockDim.x) >> 5;
    for (int64_t i = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5; i < N; i += n_warps) {
        const float4 xi = pos4[i];
        uint32_t *row = nbr + i * (int64_t)cap;
        int n = 0;
        for (int nz = -g.kimg[2]; nz <= g.kimg[2]; ++nz)
            for (int ny = -g.kimg[1]; ny <= g.kimg[1]; ++ny)
                for (int nx = -g.kimg[0]; nx <= g.kimg[0]; ++nx) {
                    const float sx = list_shift(g, 0, nx, ny, nz), sy = list_shift(g, 1, nx, ny, nz),
                                sz = list_shift(g, 2, nx, ny, nz);
                    const uint32_t code = image_code(nx, ny, nz);
                    const bool home = (nx | ny | nz) == 0;
                    for (int base = 0; base < (int)N; base += 32) {
                        const int j = base + lane;
                        bool keep = false;
                        if (j < (int)N && !(home && j == (int)i)) keep = in_list(xi, pos4[j], sx, sy, sz, g.r_list2);
                        const unsigned m = __ballot_sync(0xffffffffu, keep);
                        const int p = n + __popc(m & ((1u << lane) - 1u));
                        if (keep && p < cap) row[p] = (uint32_t)j | code;
                        n += __popc(m);
                    }
                }
        if (lane == 0) {
            count[i] = n < cap ? n : cap;
            if (n > cap) atomicMax(&flags[FLAG_MAXCOUNT], n);
        }
    }
}

// Reverse-pair index for the pair-buffer force reduction (GMNN_FORCE_PAIRBUF): rev[i][k] = slot of
// (i, -n) in the row of j, for entry k = (j, n) of row i.  The list is symmetric by construction
// (the membership predicate is exactly odd under i <-> j, n -> -n), so every entry has a partner;
// a missing one raises FLAG_REV_MISSING.  One warp per atom: each lane owns one entry of a batch of
// 32, the warp scans the partner row 32 slots at a time.
__global__ void __launch_bounds__(256)
k_build_rev(int64_t N, const uint32_t *__restrict__ nbr, const int32_t *__restrict__ count, int cap, uint16_t *rev,
            int32_t *flags, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    const int lane = threadIdx.x & 31;
    // grid-stride over atoms (one warp each): the launch is a few waves of blocks, so that the
    // every-step launches that skip_rebuild() turns into no-ops stay cheap
    const int64_t n_warps = (gridDim.x * (int64_t)blockDim.x) >> 5;
    for (int64_t i = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5; i < N; i += n_warps) {
        const int cnt = count[i];
        const uint32_t *row = nbr + i * (int64_t)cap;
        for (int k0 = 0; k0 < cnt; k0 += 32) {
            const uint32_t e_mine = k0 + lane < cnt ? row[k0 + lane] : 0u;
            int found = 0xFFFF;
            const int nk = cnt - k0 < 32 ? cnt - k0 : 32;
            for (int t = 0; t < nk; ++t) {
                const uint32_t e = __shfl_sync(0xffffffffu, e_mine, t);
                const int64_t j = e & NBR_J_MASK;
                const uint32_t img = e >> NBR_J_BITS;  // three 3-bit fields n + 4; the inverse image is 8 - field
                const uint32_t inv = (8u - (img & 7u)) | ((8u - ((img >> 3) & 7u)) << 3) | ((8u - ((img >> 6) & 7u)) << 6);
                const uint32_t target = (uint32_t)i | (inv << NBR_J_BITS);
                const uint32_t *rj = nbr + j * (int64_t)cap;
                const int cj = count[j];
                int pos = 0xFFFF;
                for (int b = 0; b < cj; b += 32) {
                    const bool hit = b + lane < cj && rj[b + lane] == target;
                    const unsigned m = __ballot_sync(0xffffffffu, hit);
                    if (m) {
                        pos = b + __ffs(m) - 1;
                        break;
                    }
                }
                if (lane == t) found = pos;
            }
            if (k0 + lane < cnt) {
                rev[i * (int64_t)cap + k0 + lane] = (uint16_t)found;
                if (found == 0xFFFF) flags[FLAG_REV_MISSING] = 1;
            }
        }
    }
}

// The same index for lists built by k_build_cells, using the runs: lane = one entry; its run r in
// row i comes from the run starts, the partner is searched only in run 26 - r of row j (about 5
// entries instead of the whole row).
__global__ void __launch_bounds__(256)
k_build_rev_runs(int64_t N, const uint32_t *__restrict__ nbr, const int32_t *__restrict__ count, int cap,
                 const uint16_t *__restrict__ runs, uint16_t *rev, int32_t *flags, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    const int lane = threadIdx.x & 31;
    // grid-stride over atoms (one warp each): the launch is a few waves of blocks, so that the
    // every-step launches that skip_rebuild() turns into no-ops stay cheap
    const int64_t n_warps = (gridDim.x * (int64_t)blockDim.x) >> 5;
    for (int64_t i = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5; i < N; i += n_warps) {
        const int cnt = count[i];
        const uint32_t *row = nbr + i * (int64_t)cap;
        const int run_lo = (int)runs[i * RUNS_PITCH + lane];  // starts of runs 0..31
        const int run_hi = lane + 32 < 54 ? (int)runs[i * RUNS_PITCH + 32 + lane] : 0x7fffffff;  // runs 32..53
        for (int k0 = 0; k0 < cnt; k0 += 32) {
            const int k = k0 + lane;
            int r = -1;  // run of slot k: number of run starts <= k, minus one
    #pragma unroll
            for (int q = 0; q < 32; ++q) r += __shfl_sync(0xffffffffu, run_lo, q) <= k ? 1 : 0;
#pragma unroll
            for (int q = 0; q < 22; ++q) r += __shfl_sync(0xffffffffu, run_hi, q) <= k ? 1 : 0;
            if (k < cnt) {
                const uint32_t e = row[k];
                const int64_t j = e & NBR_J_MASK;
                const uint32_t img = e >> NBR_J_BITS;
                const uint32_t inv = (8u - (img & 7u)) | ((8u - ((img >> 3) & 7u)) << 3) | ((8u - ((img >> 6) & 7u)) << 6);
                const uint32_t target = (uint32_t)i | (inv << NBR_J_BITS);
                const uint32_t *rj = nbr + j * (int64_t)cap;
                const int rr = (r / 27) * 27 + 26 - r % 27;  // same part, mirrored cell
                const int s0 = runs[j * RUNS_PITCH + rr], s1 = runs[j * RUNS_PITCH + rr + 1];
                int found = 0xFFFF;
                for (int t = s0; t < s1; ++t)
                    if (rj[t] == target) {
                        found = t;
                        break;
                    }
                rev[i * (int64_t)cap + k] = (uint16_t)found;
                if (found == 0xFFFF) flags[FLAG_REV_MISSING] = 1;
            }
        }
    }
}

// ---- rows of the MLP stage for per-species weight sets (gmnn_internal.h: mrow, row_atom) ---------------
// mrow[k] = seg_row0[z_k] + number of internal atoms before k with the same species: a stable counting
// sort by species of the cell-ordered atoms, so rows keep the spatial order inside a species segment and
// the assignment is a pure function of the positions (bit-reproducible).  Three small kernels per rebuild.
struct SegRows {
    int64_t row0[MAX_SPECIES];
};

__global__ void __launch_bounds__(256)
k_species_block_count(int64_t N, const float4 *__restrict__ pos4, int32_t *sp_count, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    __shared__ int32_t c[MAX_SPECIES];
    if (threadIdx.x < MAX_SPECIES) c[threadIdx.x] = 0;
    __syncthreads();
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k < N) atomicAdd(&c[__float_as_int(pos4[k].w)], 1);  // integer: order-free
    __syncthreads();
    if (threadIdx.x < MAX_SPECIES) sp_count[blockIdx.x * (int64_t)MAX_SPECIES + threadIdx.x] = c[threadIdx.x];
}

// one thread per species: exclusive scan of its per-block counts, offset by the segment's first row
__global__ void k_species_scan(int64_t n_blocks, int32_t *sp_count, SegRows seg, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    const int z = threadIdx.x;
    if (z >= MAX_SPECIES) return;
    int64_t run = seg.row0[z];
    for (int64_t b = 0; b < n_blocks; ++b) {
        const int32_t c = sp_count[b * MAX_SPECIES + z];
        sp_count[b * MAX_SPECIES + z] = (int32_t)run;
        run += c;
    }
}

__global__ void __launch_bounds__(256)
k_species_assign(int64_t N, const float4 *__restrict__ pos4, const int32_t *__restrict__ sp_count, int32_t *mrow,
                 int32_t *row_atom, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    __shared__ int32_t wc[8][MAX_SPECIES];  // per warp, per species
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int z = k < N ? __float_as_int(pos4[k].w) : -1;
    int rank = 0;
#pragma unroll
    for (int q = 0; q < MAX_SPECIES; ++q) {
        const unsigned m = __ballot_sync(0xffffffffu, z == q);
        if (z == q) rank = __popc(m & ((1u << lane) - 1u));
        if (lane == 0) wc[wid][q] = __popc(m);
    }
    __syncthreads();
    if (z < 0) return;
    int before = 0;
    for (int w = 0; w < wid; ++w) before += wc[w][z];
    const int32_t r = sp_count[blockIdx.x * (int64_t)MAX_SPECIES + z] + before + rank;
    mrow[k] = r;
    row_atom[r] = (int32_t)k;
}

__global__ void k_finish_rebuild(int32_t *flags, const int32_t *cond, float thr2) {
    if (skip_rebuild(cond, thr2)) return;
    flags[FLAG_DISP2] = 0;
    flags[FLAG_REBUILDS] += 1;
}

static inline unsigned nblocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }
// blocks of 256 threads for a thread-per-item grid-stride kernel: at most 8 blocks per SM, so that a
// launch that skip_rebuild() turns into a no-op costs a few microseconds
static inline unsigned small_grid(int64_t n_items) {
    const int64_t want = (n_items + 255) / 256, cap = 148 * 8;
    return (unsigned)(want < cap ? (want > 0 ? want : 1) : cap);
}
// blocks of 256 threads for a warp-per-atom grid-stride kernel: at most 4 waves of 148 SMs x 8 blocks.  Measured at
// config 5 (full build / the skipped launches of one MD step): 16 waves 6.25 ms / 0.14 ms, 8: 6.37 / 0.095, 4: 6.61 / 0.074,
// 2: 7.3 / 0.064 -- at one rebuild per 20 to 50 steps 4 waves cost the least per step
static inline unsigned warp_grid(int64_t n_atoms) {
    const int64_t want = (n_atoms * 32 + 255) / 256, cap = 148 * 8 * 4;
    return (unsigned)(want < cap ? want : cap);
}

int launch_build(gmnn_system *s, const float *positions, cudaStream_t st, const int32_t *cond, float thr2,
                 bool wrap_first, float *positions_mut) {
    const int64_t N = s->N;
    const Geometry g = s->geo;
    if (wrap_first && positions_mut) {
        k_wrap<<<small_grid(3 * N), 256, 0, st>>>(N, positions_mut, g, cond, thr2);
        GMNN_LAUNCHED();
    }
    k_zero_cells<<<small_grid(s->ncells + 1), 256, 0, st>>>(s->ncells, s->cell_count, s->cell_fill, cond, thr2);
    GMNN_LAUNCHED();
    k_cell_assign<<<small_grid(N), 256, 0, st>>>(N, positions, g, s->cell_of, s->cell_count, s->flags, cond, thr2);
    GMNN_LAUNCHED();
    k_scan_cells<<<1, 1024, 0, st>>>(s->ncells, s->cell_count, s->cell_start, cond, thr2);
    GMNN_LAUNCHED();
    k_cell_fill<<<small_grid(N), 256, 0, st>>>(N, s->cell_of, s->cell_start, s->cell_fill, s->slot_tmp, cond, thr2);
    GMNN_LAUNCHED();
    k_cell_rank<<<small_grid(N), 256, 0, st>>>(N, s->slot_tmp, s->cell_of, s->cell_start, s->perm, cond, thr2);
    GMNN_LAUNCHED();
    k_gather<<<nblocks(N, 256), 256, 0, st>>>(N, positions, s->species, s->perm, s->pos4, s->xref, true, 0.f,
                                              nullptr, cond, thr2);
    GMNN_LAUNCHED();
    if (s->mrow) {  // per-species weight sets: rows of the MLP stage follow the new atom order
        SegRows seg;
        for (int z = 0; z < MAX_SPECIES; ++z) seg.row0[z] = s->seg_row0[z];
        const unsigned nb = nblocks(N, 256);
        k_species_block_count<<<nb, 256, 0, st>>>(N, s->pos4, s->sp_count, cond, thr2);
        GMNN_LAUNCHED();
        k_species_scan<<<1, 32, 0, st>>>((int64_t)nb, s->sp_count, seg, cond, thr2);
        GMNN_LAUNCHED();
        k_species_assign<<<nb, 256, 0, st>>>(N, s->pos4, s->sp_count, s->mrow, s->row_atom, cond, thr2);
        GMNN_LAUNCHED();
    }
    if (s->small_box)
        k_build_small<<<warp_grid(N), 256, 0, st>>>(N, s->pos4, g, s->nbr, s->count, s->cap, s->flags, cond, thr2);
    else
        k_build_cells<<<warp_grid(N), 256, 0, st>>>(N, s->pos4, s->cell_start, g, s->nbr, s->count, s->cap,
                                                            s->flags, cond, thr2,
                                                            s->force_mode == GMNN_FORCE_PAIRBUF ? s->runs : nullptr);
    GMNN_LAUNCHED();
    if (s->force_mode == GMNN_FORCE_PAIRBUF) {
        if (s->small_box)
            k_build_rev<<<warp_grid(N), 256, 0, st>>>(N, s->nbr, s->count, s->cap, s->rev, s->flags, cond, thr2);
        else
            k_build_rev_runs<<<warp_grid(N), 256, 0, st>>>(N, s->nbr, s->count, s->cap, s->runs, s->rev, s->flags,
                                                                   cond, thr2);
        GMNN_LAUNCHED();
    }
    k_finish_rebuild<<<1, 1, 0, st>>>(s->flags, cond, thr2);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

int launch_gather_positions(gmnn_system *s, const float *positions, cudaStream_t st, bool check_stale) {
    const float hs = 0.5f * s->skin;
    k_gather<<<nblocks(s->N, 256), 256, 0, st>>>(s->N, positions, s->species, s->perm, s->pos4, s->xref, false,
                                                 hs * hs, check_stale ? s->flags : nullptr, nullptr, 0.f);
    GMNN_LAUNCHED();
    GMNN_CUDA(cudaGetLastError());
    return GMNN_OK;
}

}  // namespace gmnn
