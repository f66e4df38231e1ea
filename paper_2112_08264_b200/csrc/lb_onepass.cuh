// lb_onepass.cuh -- the fused one-pass time step: every population crosses HBM once in and once
// out per step (608 B/node fp64, 304 B/node fp32) plus ~45 B/node of density bookkeeping.
//
// State convention (whole library): the population buffer holds h_i^k(x) = the POST-collision,
// NOT yet streamed value of the previous step.  Streaming is done by the reader ("pull"):
//     f_i^k(x,t) = h_i^k(x - c_i)            (Eq. 5, periodic PAPER.md:160)
//     f_i^k(x,t) = h_opp(i)^k(x)             if x - c_i is solid (Eq. 23-24 with u_b = 0)
// Reads are misaligned by one element in x, writes are aligned full sectors: measured on B200
// pull streams at 9.6 GLUPS where push (aligned reads, misaligned writes)
// stays at 7.6-8.2.
//
// Why the density is carried from step to step:
//   The Shan-Chen force at x needs rho^kbar at the 18 neighbours of x at the SAME time level,
//   and rho(x,t) = sum_i f_i(x,t) is only known once all 19 populations of x have been pulled.
//   Recomputing the neighbours' densities costs either a second sweep (944 B/node) or, per tile,
//   halo reads that miss in L2 (measured: 824 B/node of DRAM traffic).  Instead step t produces
//   rho(.,t+1) itself: rho(y,t+1) = sum_i h_i(y - c_i), a gather over the post-collision values
//   the CTA has just computed.  One CTA owns a TX x TY column and marches along z:
//     - post-collision values are exchanged through shared memory (16 direction planes S_i,
//       zero-padded by two nodes), each thread gathers the three in-plane partial sums
//       A_dz = sum_{i: cz_i = dz} h_i(y - c_i) of its node and pipelines them along z in
//       registers: rho(z) = (A_+1(z-1) + A_0(z)) + A_-1(z+1);
//     - contributions that cross a tile edge are NOT added into the neighbour's array (that
//       would need atomics and give an order-dependent fp sum).  Each of the four arrays
//       rho_in / rho_x / rho_y / rho_xy has exactly ONE writer per entry: the owner tile (in),
//       its x neighbour (x), its y neighbour (y), its diagonal neighbour (xy).  The reader
//       assembles rho = ((in + x) + y) + xy in that fixed order: deterministic, and every CTA
//       that needs a node's density computes the same bits;
//     - along z the chunk [z0,z1) re-collides planes z0-1 and z1 (without storing them) so
//       that no partial sums cross chunk boundaries: 2/zc extra reads.
//   rho(t) for the tile and its one-node halo lives in a shared-memory ring of four planes.
//   u' needs j of BOTH components before either is collided (S4): the blue populations are
//   pulled once for their moments, then again (L1/L2 hits) for their collision, so that only
//   19 values are live at a time (<= 128 registers, two 256-thread CTAs per SM).
#pragma once
#include "lb_lattice.cuh"

namespace lb {

constexpr unsigned OP_SOLID_BIT = 1u << 31;

// the four single-writer density arrays (both components each; comp stride s_*)
template <typename T>
struct RhoView {
    T* in;  long long s_in;     // [k][NP]                              node n
    T* x;   long long s_x;      // [k][z][tile_y][tile_x][side][TY]     nodes with x_local in {0, TX-1}
    T* y;   long long s_y;      // [k][z][tile_y][side][nx]             nodes with y_local in {0, TY-1}
    T* xy;  long long s_xy;     // [k][z][tile_y][tile_x][4]            tile corners
};

// index of direction i in the shared exchange planes (directions with an in-plane offset)
__host__ __device__ constexpr int sidx(int i) { return i <= 4 ? i - 1 : i - 3; }
__host__ __device__ constexpr bool dir_local(int i) { return dir_cx(i) == 0 && dir_cy(i) == 0; }

template <typename T, int TX, int TY>
constexpr size_t onepass_smem_bytes() {
    return sizeof(T) * (size_t(8) * (TX + 2) * (TY + 2) + size_t(16) * (TX + 4) * (TY + 4));
}

template <typename T, bool HAS_SOLID, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 2)
k_step_pull(const T* __restrict__ h, T* __restrict__ g, const unsigned* __restrict__ links,
            const RhoView<T> ri, const RhoView<T> ro, long long NP, int nx, int ny, int nz, int zc,
            T om_r, T om_b, T G) {
    constexpr int NT = TX * TY;
    constexpr int RW = TX + 2, RH = TY + 2, RS = RW * RH;      // density ring plane: tile + 1 halo
    constexpr int PW = TX + 4, PH = TY + 4, PS = PW * PH;      // exchange plane: tile + 2 zero padding
    constexpr int NHALO = 2 * RW + 2 * TY;
    static_assert(NHALO <= NT, "one halo node per thread at most");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* ring = reinterpret_cast<T*>(smem_raw);                  // [4][2][RS]
    T* S = ring + 8 * RS;                                      // [16][PS]

    const int t = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    const int ntx = nx / TX, nty = ny / TY;
    const int btx = blockIdx.x, bty = blockIdx.y;
    const int x = btx * TX + tx, y = bty * TY + ty;
    const int z0 = blockIdx.z * zc;
    const int z1 = min(z0 + zc, nz);
    const long long pl = (long long)nx * ny;
    const long long psx = (long long)nty * ntx * 2 * TY, psy = (long long)nty * 2 * nx, psxy = (long long)nty * ntx * 4;

    for (int a = t; a < 16 * PS; a += NT) S[a] = T(0);         // padding stays zero for the whole kernel

    // periodic neighbours in x and y (element offsets within a plane)
    const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
    const int ys[3] = {nx * (y == 0 ? ny - 1 : y - 1), nx * y, nx * (y == ny - 1 ? 0 : y + 1)};
    const int own_xy = ys[1] + x;
    const int own_r = (ty + 1) * RW + tx + 1;
    const int own_p = (ty + 2) * PW + tx + 2;
    const bool own_ex = (tx == 0 || tx == TX - 1), own_ey = (ty == 0 || ty == TY - 1);
    const int own_ox = ((bty * ntx + btx) * 2 + (tx != 0)) * TY + ty;
    const int own_oy = (bty * 2 + (ty != 0)) * nx + x;
    const int own_oxy = (bty * ntx + btx) * 4 + (ty != 0) * 2 + (tx != 0);

    // the halo node this thread assembles (ring) and exports to (tile-relative hx in [-1,TX], hy in [-1,TY])
    const bool has_halo = t < NHALO;
    int halo_in = 0, halo_r = 0, halo_p = 0, halo_ox = 0, halo_oy = 0, halo_oxy = 0;
    bool halo_ex = false, halo_ey = false;
    if (has_halo) {
        int hx, hy;
        if (t < RW) { hx = t - 1; hy = -1; }
        else if (t < 2 * RW) { hx = t - RW - 1; hy = TY; }
        else if (t < 2 * RW + TY) { hx = -1; hy = t - 2 * RW; }
        else { hx = TX; hy = t - 2 * RW - TY; }
        const int otx = hx < 0 ? (btx == 0 ? ntx - 1 : btx - 1) : (hx >= TX ? (btx == ntx - 1 ? 0 : btx + 1) : btx);
        const int oty = hy < 0 ? (bty == 0 ? nty - 1 : bty - 1) : (hy >= TY ? (bty == nty - 1 ? 0 : bty + 1) : bty);
        const int lx = hx < 0 ? TX - 1 : (hx >= TX ? 0 : hx);
        const int ly = hy < 0 ? TY - 1 : (hy >= TY ? 0 : hy);
        const int gx = otx * TX + lx, gy = oty * TY + ly;
        halo_in = gy * nx + gx;
        halo_r = (hy + 1) * RW + hx + 1;
        halo_p = (hy + 2) * PW + hx + 2;
        halo_ex = (lx == 0 || lx == TX - 1);
        halo_ey = (ly == 0 || ly == TY - 1);
        halo_ox = ((oty * ntx + otx) * 2 + (lx != 0)) * TY + ly;
        halo_oy = (oty * 2 + (ly != 0)) * nx + gx;
        halo_oxy = (oty * ntx + otx) * 4 + (ly != 0) * 2 + (lx != 0);
    }
    // which single-writer array this CTA's contribution to its halo node goes to
    const bool halo_col = has_halo && t >= 2 * RW;                                    // hx outside, hy inside
    const bool halo_corner = has_halo && t < 2 * RW && (t % RW == 0 || t % RW == RW - 1);

    auto wrapz = [&](int p) { p %= nz; return p < 0 ? p + nz : p; };

    // rho(t) of plane p at the own node and at the halo node: ((in + x) + y) + xy
    auto ring_load = [&](int p, T (&v)[4]) {
        const long long zl = wrapz(p);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T a = __ldg(ri.in + k * ri.s_in + zl * pl + own_xy);
            if (own_ex) a += __ldg(ri.x + k * ri.s_x + zl * psx + own_ox);
            if (own_ey) a += __ldg(ri.y + k * ri.s_y + zl * psy + own_oy);
            if (own_ex && own_ey) a += __ldg(ri.xy + k * ri.s_xy + zl * psxy + own_oxy);
            v[k] = a;
            if (has_halo) {
                T b = __ldg(ri.in + k * ri.s_in + zl * pl + halo_in);
                if (halo_ex) b += __ldg(ri.x + k * ri.s_x + zl * psx + halo_ox);
                if (halo_ey) b += __ldg(ri.y + k * ri.s_y + zl * psy + halo_oy);
                if (halo_ex && halo_ey) b += __ldg(ri.xy + k * ri.s_xy + zl * psxy + halo_oxy);
                v[2 + k] = b;
            }
        }
    };
    auto ring_store = [&](int p, const T (&v)[4]) {
        const int slot = (p - z0 + 2) & 3;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            ring[(slot * 2 + k) * RS + own_r] = v[k];
            if (has_halo) ring[(slot * 2 + k) * RS + halo_r] = v[2 + k];
        }
    };

    {
        T v[4];
#pragma unroll 1
        for (int p = z0 - 2; p <= z0; ++p) { ring_load(p, v); ring_store(p, v); }
    }
    __syncthreads();

    // z pipelines of the density partial sums: [k][0] = A_+1(z-1) + A_0(z) so far, [k][1] = A_+1(z)
    T own_acc[2][2] = {{T(0), T(0)}, {T(0), T(0)}};
    T halo_acc[2][2] = {{T(0), T(0)}, {T(0), T(0)}};

#pragma unroll 1
    for (int z = z0 - 1; z <= z1; ++z) {
        const int zt = wrapz(z - 1);                             // plane index of the density target
        const long long zoff[3] = {zt * pl, wrapz(z) * pl, wrapz(z + 1) * pl};
        const long long n = zoff[1] + own_xy;
        const bool store_h = z >= z0 && z < z1;                 // planes z0-1 and z1 are re-collided only
        const bool store_rho = z - 1 >= z0;                     // target plane z-1 (always < z1 here)
        const int s0 = (z - z0 + 2) & 3;                        // ring slot of plane z
        unsigned lk = 0;
        if (HAS_SOLID) lk = __ldg(links + n);
        const bool fluid = !HAS_SOLID || !(lk & OP_SOLID_BIT);  // nothing happens inside a particle

        // pull the 19 populations of component k arriving at this node (Eq. 5 / Eq. 23-24)
        auto pull = [&](int k, T (&fk)[Q]) {
            const T* base = h + (long long)(k * Q) * NP;
#pragma unroll
            for (int i = 0; i < Q; ++i) {
                const T* src = base + (long long)i * NP + zoff[1 - dir_cz(i)] + ys[1 - dir_cy(i)] + xs[1 - dir_cx(i)];
                if (HAS_SOLID && i > 0 && (lk >> dir_opp(i) & 1u)) src = base + (long long)dir_opp(i) * NP + n;
                fk[i] = __ldg(src);
            }
        };
        // exchange the post-collision values and gather this step's contribution to rho(t+1)
        auto publish = [&](const T (&fk)[Q]) {
#pragma unroll
            for (int i = 1; i < Q; ++i)
                if (!dir_local(i)) S[sidx(i) * PS + own_p] = fk[i];
        };
        auto gather = [&](int k, const T (&fk)[Q]) {
            T a[3] = {T(0), T(0), T(0)};                         // index cz + 1
#pragma unroll
            for (int i = 0; i < Q; ++i)
                a[dir_cz(i) + 1] += dir_local(i) ? fk[i] : S[sidx(i) * PS + own_p - dir_cy(i) * PW - dir_cx(i)];
            if (HAS_SOLID) {                                     // bounced-back arrivals come from this node itself
#pragma unroll
                for (int i = 1; i < Q; ++i)
                    if (lk >> dir_opp(i) & 1u) a[1] += fk[dir_opp(i)];
            }
            const T out = own_acc[k][0] + a[0];
            own_acc[k][0] = own_acc[k][1] + a[1];
            own_acc[k][1] = a[2];
            if (store_rho) ro.in[k * ro.s_in + zoff[0] + own_xy] = out;
            if (has_halo) {
                T b[3] = {T(0), T(0), T(0)};
#pragma unroll
                for (int i = 1; i < Q; ++i)
                    if (!dir_local(i)) b[dir_cz(i) + 1] += S[sidx(i) * PS + halo_p - dir_cy(i) * PW - dir_cx(i)];
                const T hout = halo_acc[k][0] + b[0];
                halo_acc[k][0] = halo_acc[k][1] + b[1];
                halo_acc[k][1] = b[2];
                if (store_rho) {
                    if (halo_corner) ro.xy[k * ro.s_xy + zt * psxy + halo_oxy] = hout;
                    else if (halo_col) ro.x[k * ro.s_x + zt * psx + halo_ox] = hout;
                    else ro.y[k * ro.s_y + zt * psy + halo_oy] = hout;
                }
            }
        };

        T fk[Q];
        T rb = T(0), ux = T(0), uy = T(0), uz = T(0);
        T eb[3] = {T(0), T(0), T(0)};
        if (fluid) {
            T jb[3], jr[3], rr;
            pull(1, fk);
            moments19<T>(fk, rb, jb[0], jb[1], jb[2]);
            pull(0, fk);
            moments19<T>(fk, rr, jr[0], jr[1], jr[2]);
            const T den = om_r * rr + om_b * rb;                 // S4
            const T inv = den != T(0) ? T(1) / den : T(0);
            ux = (om_r * jr[0] + om_b * jb[0]) * inv;
            uy = (om_r * jr[1] + om_b * jb[1]) * inv;
            uz = (om_r * jr[2] + om_b * jb[2]) * inv;
            // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6); a solid neighbour counts 0 (S7)
            T gr[3] = {T(0), T(0), T(0)}, gb[3] = {T(0), T(0), T(0)};
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm = (s0 - pair_cz(p)) & 3;
                const int op = own_r + pair_cy(p) * RW + pair_cx(p), om = own_r - pair_cy(p) * RW - pair_cx(p);
                T bp = ring[(sp * 2 + 1) * RS + op], bm = ring[(sm * 2 + 1) * RS + om];
                T rp = ring[(sp * 2 + 0) * RS + op], rm = ring[(sm * 2 + 0) * RS + om];
                if (HAS_SOLID) {
                    if (lk >> (2 * p + 1) & 1u) { bp = T(0); rp = T(0); }
                    if (lk >> (2 * p + 2) & 1u) { bm = T(0); rm = T(0); }
                }
                const T db = w_pair<T>(p) * (bp - bm);
                const T dr = w_pair<T>(p) * (rp - rm);
                if (pair_cx(p)) { gr[0] += T(pair_cx(p)) * db; gb[0] += T(pair_cx(p)) * dr; }
                if (pair_cy(p)) { gr[1] += T(pair_cy(p)) * db; gb[1] += T(pair_cy(p)) * dr; }
                if (pair_cz(p)) { gr[2] += T(pair_cz(p)) * db; gb[2] += T(pair_cz(p)) * dr; }
            }
            eb[0] = ux - G * gb[0]; eb[1] = uy - G * gb[1]; eb[2] = uz - G * gb[2];
            collide19<T>(fk, rr, T(1) - om_r, ux, uy, uz, ux - G * gr[0], uy - G * gr[1], uz - G * gr[2]);
            if (store_h) {
#pragma unroll
                for (int i = 0; i < Q; ++i) g[(long long)i * NP + n] = fk[i];
            }
        } else {
#pragma unroll
            for (int i = 0; i < Q; ++i) fk[i] = T(0);
        }
        publish(fk);
        __syncthreads();
        gather(0, fk);
        __syncthreads();

        T rv[4];
        const bool fill = z < z1;                                // plane z+2 is needed by iteration z+1
        if (fill) ring_load(z + 2, rv);
        if (fluid) {
            pull(1, fk);
            collide19<T>(fk, rb, T(1) - om_b, ux, uy, uz, eb[0], eb[1], eb[2]);
            if (store_h) {
#pragma unroll
                for (int i = 0; i < Q; ++i) g[(long long)(Q + i) * NP + n] = fk[i];
            }
        }
        publish(fk);
        if (fill) ring_store(z + 2, rv);
        __syncthreads();
        gather(1, fk);
        __syncthreads();
    }
}

}  // namespace lb
