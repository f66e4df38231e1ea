// lb_onepass.cuh -- the fused one-pass time step: every population crosses HBM once in and once
// out per step (608 B/node fp64, 304 B/node fp32); the density field is never stored.
//
// Why it is shaped like this:
//   The Shan-Chen force at x needs rho^kbar at the 18 neighbours of x AT THE SAME TIME LEVEL,
//   and rho is a sum over all 19 populations of a node (Eq. 6).  A separate density pass
//   re-reads all 38 populations (944 B/node, <= 64 % of roofline).  Here one CTA owns a
//   TX x TY column of the box and marches along z.  A ring of four density planes
//   (tile + one-node halo, both components) lives in shared memory:
//     phase A(z+1): each thread streams the 38 populations of its node in plane z+1, sums
//                   rho^k (-> ring) and j^k (-> registers, used one iteration later); the first
//                   2*(TX+2)+2*TY threads also sum rho^k of one halo node each.  Halo lines are
//                   the neighbouring CTA's own lines: they come from L2 (measured 32 TB/s on
//                   B200, 5x HBM), not from HBM.
//     __syncthreads
//     phase B(z):   u' from the carried j^k, force from the ring (36 LDS), then per component:
//                   re-read the 19 populations of plane z (L1/L2 hits: they were streamed in
//                   by phase A one iteration ago), collide (lb_lattice.cuh), push-stream with
//                   periodic wrap / halfway bounce-back.
//   One barrier per plane: slot(z+2) == slot(z-2) was last read before the previous barrier.
//   Registers: one component (19 values) live at a time + 6 carried momenta -> <= 128 regs in
//   fp64, two 256-thread CTAs per SM.
#pragma once
#include "lb_lattice.cuh"

namespace lb {

constexpr unsigned OP_SOLID_BIT = 1u << 31;

template <typename T> __device__ __forceinline__ T ld_stream(const T* p) { return __ldg(p); }

template <typename T, bool HAS_SOLID, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 2)
k_step_onepass(const T* __restrict__ f, T* __restrict__ g, const unsigned* __restrict__ links,
               long long NP, int nx, int ny, int nz, int zc, T om_r, T om_b, T G) {
    constexpr int RW = TX + 2, RH = TY + 2, RS = RW * RH;
    constexpr int NHALO = 2 * RW + 2 * TY;
    static_assert(NHALO <= TX * TY, "one halo node per thread at most");
    __shared__ T ring[4][2][RS];

    const int t = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    const int x = blockIdx.x * TX + tx, y = blockIdx.y * TY + ty;
    const int z0 = blockIdx.z * zc;
    const int z1 = min(z0 + zc, nz);
    const long long pl = (long long)nx * ny;

    // periodic neighbours in x and y (element offsets within a plane)
    const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
    const int ys[3] = {nx * (y == 0 ? ny - 1 : y - 1), nx * y, nx * (y == ny - 1 ? 0 : y + 1)};
    const int own_xy = ys[1] + x;
    const int own_r = (ty + 1) * RW + tx + 1;

    // the halo node this thread sums (tile-relative hx in [-1,TX], hy in [-1,TY])
    int halo_xy = -1, halo_r = 0;
    if (t < NHALO) {
        int hx, hy;
        if (t < RW) { hx = t - 1; hy = -1; }
        else if (t < 2 * RW) { hx = t - RW - 1; hy = TY; }
        else if (t < 2 * RW + TY) { hx = -1; hy = t - 2 * RW; }
        else { hx = TX; hy = t - 2 * RW - TY; }
        int gx = blockIdx.x * TX + hx, gy = blockIdx.y * TY + hy;
        gx = gx < 0 ? gx + nx : (gx >= nx ? gx - nx : gx);
        gy = gy < 0 ? gy + ny : (gy >= ny ? gy - ny : gy);
        halo_xy = gy * nx + gx;
        halo_r = (hy + 1) * RW + hx + 1;
    }

    // phase A: densities of plane p (tile + halo) into the ring; momenta of the own node out
    auto density_plane = [&](int p, T (&j)[6]) {
        const int zl = p < 0 ? p + nz : (p >= nz ? p - nz : p);
        const int slot = (p - z0 + 1) & 3;
        const T* base = f + zl * pl;
        {
            const T* q = base + own_xy;
            T fk[Q];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
#pragma unroll
                for (int i = 0; i < Q; ++i) fk[i] = ld_stream(q + (long long)(k * Q + i) * NP);
                T r;
                moments19<T>(fk, r, j[3 * k], j[3 * k + 1], j[3 * k + 2]);
                ring[slot][k][own_r] = r;
            }
        }
        if (halo_xy >= 0) {
            const T* q = base + halo_xy;
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                T r = ld_stream(q + (long long)(k * Q) * NP);
#pragma unroll
                for (int i = 1; i < Q; ++i) r += ld_stream(q + (long long)(k * Q + i) * NP);
                ring[slot][k][halo_r] = r;
            }
        }
    };

    T jc[6], jn[6];
    density_plane(z0 - 1, jn);
    density_plane(z0, jc);

    for (int z = z0; z < z1; ++z) {
        density_plane(z + 1, jn);
        __syncthreads();

        const long long zoff[3] = {(z == 0 ? nz - 1 : z - 1) * pl, z * pl, (z == nz - 1 ? 0 : z + 1) * pl};
        const long long n = zoff[1] + own_xy;
        unsigned lk = 0;
        if (HAS_SOLID) lk = links[n];
        if (!HAS_SOLID || !(lk & OP_SOLID_BIT)) {            // nothing happens inside a particle
            const int s0 = (z - z0 + 1) & 3;                  // slot of plane z; z-1 -> s0-1, z+1 -> s0+1
            const T rr = ring[s0][0][own_r], rb = ring[s0][1][own_r];
            const T den = om_r * rr + om_b * rb;              // S4
            const T inv = den != T(0) ? T(1) / den : T(0);
            const T ux = (om_r * jc[0] + om_b * jc[3]) * inv;
            const T uy = (om_r * jc[1] + om_b * jc[4]) * inv;
            const T uz = (om_r * jc[2] + om_b * jc[5]) * inv;
            // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6, S7), both components at once
            T gr[3] = {T(0), T(0), T(0)}, gb[3] = {T(0), T(0), T(0)};
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm = (s0 - pair_cz(p)) & 3;
                const int op = own_r + pair_cy(p) * RW + pair_cx(p), om = own_r - pair_cy(p) * RW - pair_cx(p);
                const T db = w_pair<T>(p) * (ring[sp][1][op] - ring[sm][1][om]);
                const T dr = w_pair<T>(p) * (ring[sp][0][op] - ring[sm][0][om]);
                if (pair_cx(p)) { gr[0] += T(pair_cx(p)) * db; gb[0] += T(pair_cx(p)) * dr; }
                if (pair_cy(p)) { gr[1] += T(pair_cy(p)) * db; gb[1] += T(pair_cy(p)) * dr; }
                if (pair_cz(p)) { gr[2] += T(pair_cz(p)) * db; gb[2] += T(pair_cz(p)) * dr; }
            }
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const T* q = f + n + (long long)(k * Q) * NP;
                T* o = g + (long long)(k * Q) * NP;
                T fk[Q];
#pragma unroll
                for (int i = 0; i < Q; ++i) fk[i] = ld_stream(q + (long long)i * NP);
                const T* gk = k == 0 ? gr : gb;
                collide19<T>(fk, k == 0 ? rr : rb, T(1) - (k == 0 ? om_r : om_b), ux, uy, uz,
                             ux - G * gk[0], uy - G * gk[1], uz - G * gk[2]);
#pragma unroll
                for (int i = 0; i < Q; ++i) {
                    if (HAS_SOLID && (lk >> i & 1u)) {        // Eq. 23-24, u_b = 0
                        o[(long long)dir_opp(i) * NP + n] = fk[i];
                    } else {                                   // Eq. 5, periodic
                        o[(long long)i * NP + zoff[dir_cz(i) + 1] + ys[dir_cy(i) + 1] + xs[dir_cx(i) + 1]] = fk[i];
                    }
                }
            }
        }
#pragma unroll
        for (int a = 0; a < 6; ++a) jc[a] = jn[a];
    }
}

}  // namespace lb
