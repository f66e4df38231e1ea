// lb_lattice.cuh -- D3Q19 constants and the per-node collision arithmetic of the CUDA path.
// (The CPU oracle has its own, separately written tables; nothing here is shared with it.)
//
// Direction numbering = include/lb.h (reading S1).  Directions come in opposite pairs
// (2p+1, 2p+2), p = 0..8, which lets a pair share its (c.u)^2 term.
#pragma once
#include <cuda_runtime.h>

namespace lb {

constexpr int Q = 19;
constexpr int NPOP = 2 * Q;          // two components

// Plane of population (component k, direction i) inside a population buffer [NPOP][NP]: direction-major, the two
// components of a direction adjacent, so that one TMA box (x, y, z, 2 planes) brings both (lb_tma.cuh).  Private to
// the library: the ABI's order [k][i] is produced by the transfer calls.
__host__ __device__ constexpr int pop_plane(int k, int i) { return 2 * i + k; }

// c_i of the ODD member of pair p (direction 2p+1); the even member is its negative.
__host__ __device__ constexpr int pair_cx(int p) { return (p == 0 || p == 3 || p == 4 || p == 5 || p == 6) ? 1 : 0; }
__host__ __device__ constexpr int pair_cy(int p) { return (p == 1 || p == 3 || p == 7 || p == 8) ? 1 : (p == 4 ? -1 : 0); }
__host__ __device__ constexpr int pair_cz(int p) { return (p == 2 || p == 5 || p == 7) ? 1 : ((p == 6 || p == 8) ? -1 : 0); }
// pairs: 0:(+x) 1:(+y) 2:(+z) 3:(+x+y) 4:(+x-y) 5:(+x+z) 6:(+x-z) 7:(+y+z) 8:(+y-z)

__host__ __device__ constexpr int dir_cx(int i) { return i == 0 ? 0 : ((i & 1) ? pair_cx((i - 1) / 2) : -pair_cx((i - 2) / 2)); }
__host__ __device__ constexpr int dir_cy(int i) { return i == 0 ? 0 : ((i & 1) ? pair_cy((i - 1) / 2) : -pair_cy((i - 2) / 2)); }
__host__ __device__ constexpr int dir_cz(int i) { return i == 0 ? 0 : ((i & 1) ? pair_cz((i - 1) / 2) : -pair_cz((i - 2) / 2)); }
__host__ __device__ constexpr int dir_opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }

// Lattice weights: 1/3 rest, 1/18 axis (pairs 0-2), 1/36 diagonal (pairs 3-8).
template <typename T> __host__ __device__ constexpr T w_rest() { return T(1.0 / 3.0); }
template <typename T> __host__ __device__ constexpr T w_pair(int p) { return p < 3 ? T(1.0 / 18.0) : T(1.0 / 36.0); }

// c_p . v for the odd member of pair p, written without the multiplications by 0 and 1 that IEEE arithmetic does not
// let the compiler drop (0 * x and 0 + x are not x for infinities / -0): p is a compile-time constant after unrolling.
template <typename T>
__device__ __forceinline__ T cdot(int p, T x, T y, T z) {
    return p == 0 ? x : p == 1 ? y : p == 2 ? z : p == 3 ? x + y : p == 4 ? x - y : p == 5 ? x + z : p == 6 ? x - z : p == 7 ? y + z : y - z;
}

// rho = sum_i f_i and j = sum_i f_i c_i of one component (Eq. 6-7).
template <typename T>
__device__ __forceinline__ void moments19(const T (&f)[Q], T& rho, T& jx, T& jy, T& jz) {
    T r = f[0], d[9];
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        r += f[2 * p + 1] + f[2 * p + 2];
        d[p] = f[2 * p + 1] - f[2 * p + 2];
    }
    rho = r;
    jx = (((d[0] + d[3]) + d[4]) + d[5]) + d[6];       // pairs with c_x = +1
    jy = (((d[1] + d[3]) - d[4]) + d[7]) + d[8];       // c_y = +1, +1, -1, +1, +1
    jz = (((d[2] + d[5]) - d[6]) + d[7]) - d[8];       // c_z = +1, +1, -1, +1, -1
}

// BGK collision with exact-difference forcing (Eq. 1; Eq. 10, PAPER.md:338-342;
// reading S5), in place:
//   f*_i = (1-om) f_i + om feq_i(rho,u) + feq_i(rho,u+du) - feq_i(rho,u)
//        = omc f_i + [ feq_i(rho,ue) - omc feq_i(rho,u) ],   omc = 1-om, ue = u+du.
// With s(v) = 1 - 1.5 v.v + 4.5 (c.v)^2 the pair (i, opp i) shares s; they differ in +-3 c.v.
// omc is a run-time value; nothing here specialises tau = 1.
template <typename T>
__device__ __forceinline__ void collide19(T (&f)[Q], T rho, T omc, T ux, T uy, T uz, T ex, T ey, T ez) {
    const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    const T ae = T(1) - T(1.5) * (ex * ex + ey * ey + ez * ez);
    f[0] = omc * f[0] + w_rest<T>() * rho * (ae - omc * a0);
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        const T cu = cdot<T>(p, ux, uy, uz);
        const T ce = cdot<T>(p, ex, ey, ez);
        const T wr = w_pair<T>(p) * rho;
        const T s0 = a0 + T(4.5) * cu * cu;
        const T se = ae + T(4.5) * ce * ce;
        const T sym = wr * (se - omc * s0);
        const T asym = (T(3) * wr) * (ce - omc * cu);
        f[2 * p + 1] = omc * f[2 * p + 1] + (sym + asym);
        f[2 * p + 2] = omc * f[2 * p + 2] + (sym - asym);
    }
}

// The same collision, handing the post-collision values to the caller pair by pair (`rest(h_0)`, then `pair(p, h_{2p+1},
// h_{2p+2})` for p = 0..8) and keeping nothing: what the caller does with a pair (store, gather) interleaves with the
// arithmetic of the next ones, and the inputs' registers die as the loop proceeds.
template <typename T, typename Rest, typename Pair>
__device__ __forceinline__ void collide19_pairs(const T (&f)[Q], T rho, T omc, T ux, T uy, T uz, T ex, T ey, T ez, Rest rest, Pair pair) {
    const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    const T ae = T(1) - T(1.5) * (ex * ex + ey * ey + ez * ez);
    rest(omc * f[0] + w_rest<T>() * rho * (ae - omc * a0));
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        const T cu = cdot<T>(p, ux, uy, uz);
        const T ce = cdot<T>(p, ex, ey, ez);
        const T wr = w_pair<T>(p) * rho;
        const T s0 = a0 + T(4.5) * cu * cu;
        const T se = ae + T(4.5) * ce * ce;
        const T sym = wr * (se - omc * s0);
        const T asym = (T(3) * wr) * (ce - omc * cu);
        pair(p, omc * f[2 * p + 1] + (sym + asym), omc * f[2 * p + 2] + (sym - asym));
    }
}

// B_i of the colour-gradient perturbation: -2/9 rest, 1/54 axis, 1/27 diagonal.
template <typename T> __host__ __device__ constexpr T cg_b_rest() { return T(-2.0 / 9.0); }
template <typename T> __host__ __device__ constexpr T cg_b_pair(int p) { return p < 3 ? T(1.0 / 54.0) : T(1.0 / 27.0); }

// Colour-gradient collision (readings C1-C6 of DESIGN.md section 3) for ONE component of a node, handed out
// pair by pair like collide19_pairs.  fs = sum_k f_i^k (the recolouring works on the colour-blind total), rt = rho,
// x_own = rho^k / rho, (ux, uy, uz) by Eq. 7, om the local relaxation frequency, amp = (A / 2) |grad Theta| with
// A = (9/4) sigma om (Eq. 17, 19), (gx, gy, gz) = grad Theta, ig2 = 1 / |grad|^2 and ign = 1 / |grad| (0 without a gradient),
// rcs = +- beta rho^1 rho^2 / rho (Eq. 20: + for the first component, Eq. 21: - for the second).
template <typename T, typename Rest, typename Pair>
__device__ __forceinline__ void collide19_cg_pairs(const T (&fs)[Q], T rt, T x_own, T om, T ux, T uy, T uz, T amp, T gx, T gy, T gz,
                                                    T ig2, T ign, T rcs, Rest rest, Pair pair) {
    const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    const T omc = T(1) - om, amp2 = T(2) * amp;        // both components carry the same perturbation
    rest(x_own * (omc * fs[0] + om * w_rest<T>() * rt * a0 - amp2 * cg_b_rest<T>()));      // cos(phi_0) = 0: no recolouring term
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        const T cu = cdot<T>(p, ux, uy, uz), cg = cdot<T>(p, gx, gy, gz);
        const T wr = om * (w_pair<T>(p) * rt);
        const T s0 = a0 + T(4.5) * cu * cu;
        const T pert = amp2 * (w_pair<T>(p) * cg * cg * ig2 - cg_b_pair<T>(p));             // Eq. 17: the same for i and opp(i)
        const T recol = rcs * w_pair<T>(p) * cg * ign * (p < 3 ? T(1) : T(0.70710678118654752440));   // cos(phi_i) = c_i.grad / (|c_i| |grad|)
        const T f1 = omc * fs[2 * p + 1] + wr * (s0 + T(3) * cu) + pert;
        const T f2 = omc * fs[2 * p + 2] + wr * (s0 - T(3) * cu) + pert;
        pair(p, x_own * f1 + recol, x_own * f2 - recol);                                    // Eq. 20-21
    }
}

// Eq. 10 for all 19 directions.
template <typename T>
__device__ __forceinline__ void equilibrium19(T (&f)[Q], T rho, T ux, T uy, T uz) {
    const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
    f[0] = w_rest<T>() * rho * a0;
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        const T cu = cdot<T>(p, ux, uy, uz);
        const T wr = w_pair<T>(p) * rho;
        const T s0 = a0 + T(4.5) * cu * cu;
        f[2 * p + 1] = wr * (s0 + T(3) * cu);
        f[2 * p + 2] = wr * (s0 - T(3) * cu);
    }
}

}  // namespace lb
