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
//   the CTA has just computed.  One CTA owns a 32 x TY column (one warp per row) and marches
//   along z.  The gather is separable:
//     x:  row sums  U0/Up/Um[dz] = h(x) + h(x-1) + h(x+1)  over the directions with cy = 0/+1/-1,
//         cz = dz, by warp shuffles;
//     y:  A_dz(y) = U0[dz](y) + Up[dz](y-1) + Um[dz](y+1)  through shared memory (6 planes per
//         component);
//     z:  rho(z) = (A_+1(z-1) + A_0(z)) + A_-1(z+1)  pipelined in registers.
//   Contributions that cross a tile edge are NOT added into the neighbour's array (that would
//   need atomics and give an order-dependent fp sum).  Each of the four arrays rho_in / rho_x /
//   rho_y / rho_xy has exactly ONE writer per entry: the owner tile (in), its x neighbour (x),
//   its y neighbour (y), its diagonal neighbour (xy).  The reader assembles
//   rho = ((in + x) + y) + xy in that fixed order: deterministic, and every CTA that needs a
//   node's density computes the same bits.  Along z the chunk [z0,z1) re-collides planes z0-1
//   and z1 (without storing them) so that no partial sums cross chunk boundaries: 2/zc extra
//   reads.  rho(t) for the tile and its one-node halo lives in a shared-memory ring of four planes,
//   filled two planes ahead with cp.async.
//
// Latency hiding (two 256-thread CTAs per SM, <= 128 registers, two barriers per plane):
//   u' needs j of BOTH components before either is collided (S4), and 38 live populations do
//   not fit the register budget.  The blue populations of the NEXT plane are therefore pulled
//   with cp.async into a thread-private shared-memory stash (no registers in flight, no barrier:
//   a thread only reads its own slots); their moments and their collision stream out of the
//   stash pair by pair.  The red populations of the next plane are pulled into the one register
//   array as soon as this plane's red collision has been published.
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
    T* xy;  long long s_xy;     // [k][z][tile_y][tile_x][4]            tile corners, index 2*(y_local != 0) + (x_local != 0)
};

template <int TX, int TY>
struct OnepassLayout {
    static constexpr int NT = TX * TY;
    static constexpr int RW = TX + 2, RH = TY + 2, RS = RW * RH;       // tile + one-node frame
    static constexpr int NPX = 4 * RH, NPY = 4 * RW, NPXY = 16, NPIECE = NPX + NPY + NPXY;
    static constexpr int NEDGE = NPX + 4 * (RW - 4);                   // ring positions that have edge pieces
    // element offsets into shared memory
    static constexpr int RING = 0;                                     // [4][2][RS]   rho(t), planes z-1..z+2
    static constexpr int SU = RING + 8 * RS;                           // [2][6][RS]   Up[dz], Um[dz] per component; frame = 0
    static constexpr int STASH = SU + 12 * RS;                         // [Q][NT]      pulled blue populations of this thread
    static constexpr int STAGE = STASH + Q * NT;                       // [2][NPIECE]  edge pieces of the ring plane being filled
    static constexpr int E0 = STAGE + 2 * NPIECE;                      // [2][3][2][TY] U0[dz] of the virtual columns -1 and TX
    static constexpr int ACCR = E0 + 12 * TY;                          // [2][2][TX][2] z pipelines of the row exports
    static constexpr int ACCC = ACCR + 8 * TX;                         // [2][2][TY][2] z pipelines of the column exports
    static constexpr int TOTAL = ACCC + 8 * TY;
};

template <typename T, int TX, int TY>
constexpr size_t onepass_smem_bytes() { return sizeof(T) * size_t(OnepassLayout<TX, TY>::TOTAL); }

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gsrc) {
    const unsigned d = static_cast<unsigned>(__cvta_generic_to_shared(smem_dst));
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;\n" ::"r"(d), "l"(gsrc), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename T, bool HAS_SOLID, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 2)
k_step_pull(const T* __restrict__ h, T* __restrict__ g, const unsigned* __restrict__ links,
            const RhoView<T> ri, const RhoView<T> ro, long long NP, int nx, int ny, int nz, int zc,
            T om_r, T om_b, T G) {
    using L = OnepassLayout<TX, TY>;
    static_assert(TX == 32, "one warp per tile row: the x gather uses warp shuffles");
    constexpr int NT = L::NT, RW = L::RW, RH = L::RH, RS = L::RS;
    constexpr int NPX = L::NPX, NPY = L::NPY, NPIECE = L::NPIECE, NEDGE = L::NEDGE;
    static_assert(NPIECE <= NT && NEDGE <= NT && RS <= 2 * NT, "ring fill work must fit the CTA");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    T* ring = sm + L::RING;
    T* SU = sm + L::SU;
    T* stash = sm + L::STASH;
    T* stage = sm + L::STAGE;
    T* e0a = sm + L::E0;
    T* accr = sm + L::ACCR;
    T* accc = sm + L::ACCC;

    const int t = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    const int ntx = nx / TX, nty = ny / TY;
    const int btx = blockIdx.x, bty = blockIdx.y;
    const int x = btx * TX + tx, y = bty * TY + ty;
    const int z0 = blockIdx.z * zc;
    const int z1 = min(z0 + zc, nz);
    const long long pl = (long long)nx * ny;
    const long long psx = (long long)nty * ntx * 2 * TY, psy = (long long)nty * 2 * nx, psxy = (long long)nty * ntx * 4;
    const int btxm = btx == 0 ? ntx - 1 : btx - 1, btxp = btx == ntx - 1 ? 0 : btx + 1;
    const int btym = bty == 0 ? nty - 1 : bty - 1, btyp = bty == nty - 1 ? 0 : bty + 1;

    for (int a = t; a < L::STASH - L::SU; a += NT) SU[a] = T(0);          // the frame stays zero for the whole kernel
    for (int a = t; a < L::TOTAL - L::STAGE; a += NT) stage[a] = T(0);   // stage, e0, export pipelines

    // periodic neighbours in x and y (element offsets within a plane)
    const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
    const int ys[3] = {nx * (y == 0 ? ny - 1 : y - 1), nx * y, nx * (y == ny - 1 ? 0 : y + 1)};
    const int own_xy = ys[1] + x;
    const int own_r = (ty + 1) * RW + tx + 1;

    auto wrapz = [&](int p) { p %= nz; return p < 0 ? p + nz : p; };

    // ---- ring fill: what this thread copies for every plane ------------------------------------
    // tile-relative (rx, ry) in [-1,TX] x [-1,TY] -> owner tile, local coordinates, global x / y
    auto owner = [&](int rx, int ry, int& otx, int& oty, int& lx, int& ly) {
        otx = rx < 0 ? btxm : (rx >= TX ? btxp : btx);
        oty = ry < 0 ? btym : (ry >= TY ? btyp : bty);
        lx = rx < 0 ? TX - 1 : (rx >= TX ? 0 : rx);
        ly = ry < 0 ? TY - 1 : (ry >= TY ? 0 : ry);
    };
    int in_off[2] = {0, -1};                                             // rho_in offsets of ring positions t, t + NT
#pragma unroll
    for (int a = 0; a < 2; ++a) {
        const int pos = t + a * NT;
        if (pos < RS) {
            int otx, oty, lx, ly;
            owner(pos % RW - 1, pos / RW - 1, otx, oty, lx, ly);
            in_off[a] = (oty * TY + ly) * nx + otx * TX + lx;
        }
    }
    int piece_off = -1, piece_kind = 0;                                  // edge piece t: 0 = x, 1 = y, 2 = xy
    if (t < NPIECE) {
        int rx, ry;
        if (t < NPX) { const int c4 = t / RH; rx = c4 == 0 ? -1 : (c4 == 1 ? 0 : (c4 == 2 ? TX - 1 : TX)); ry = t % RH - 1; piece_kind = 0; }
        else if (t < NPX + NPY) { const int q = t - NPX, r4 = q / RW; ry = r4 == 0 ? -1 : (r4 == 1 ? 0 : (r4 == 2 ? TY - 1 : TY)); rx = q % RW - 1; piece_kind = 1; }
        else { const int q = t - NPX - NPY, r4 = q / 4, c4 = q % 4;
               ry = r4 == 0 ? -1 : (r4 == 1 ? 0 : (r4 == 2 ? TY - 1 : TY)); rx = c4 == 0 ? -1 : (c4 == 1 ? 0 : (c4 == 2 ? TX - 1 : TX)); piece_kind = 2; }
        int otx, oty, lx, ly;
        owner(rx, ry, otx, oty, lx, ly);
        if (piece_kind == 0) piece_off = ((oty * ntx + otx) * 2 + (lx != 0)) * TY + ly;
        else if (piece_kind == 1) piece_off = (oty * 2 + (ly != 0)) * nx + otx * TX + lx;
        else piece_off = (oty * ntx + otx) * 4 + (ly != 0) * 2 + (lx != 0);
    }
    // rho(t) of plane p: the rho_in part goes straight into the ring, the edge pieces into `stage`
    auto ring_issue = [&](int p) {
        const long long zl = wrapz(p);
        const int slot = (p - z0 + 2) & 3;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T* dst = ring + (slot * 2 + k) * RS;
            cp_async<sizeof(T)>(dst + t, ri.in + k * ri.s_in + zl * pl + in_off[0]);
            if (in_off[1] >= 0) cp_async<sizeof(T)>(dst + t + NT, ri.in + k * ri.s_in + zl * pl + in_off[1]);
            if (piece_off >= 0) {
                const T* src = piece_kind == 0 ? ri.x + k * ri.s_x + zl * psx
                             : (piece_kind == 1 ? ri.y + k * ri.s_y + zl * psy : ri.xy + k * ri.s_xy + zl * psxy);
                cp_async<sizeof(T)>(stage + k * NPIECE + t, src + piece_off);
            }
        }
        cp_async_commit();
    };
    // rho = ((in + x) + y) + xy on the ring positions that have edge pieces (after a barrier)
    auto ring_assemble = [&](int p) {
        if (t >= NEDGE) return;
        const int slot = (p - z0 + 2) & 3;
        if (t < NPX) {
            const int c4 = t / RH, ryi = t % RH;
            const int rx = c4 == 0 ? -1 : (c4 == 1 ? 0 : (c4 == 2 ? TX - 1 : TX));
            const int pos = ryi * RW + rx + 1;
            const bool hasy = ryi < 2 || ryi >= TY;
            const int r4 = ryi < 2 ? ryi : ryi - (TY - 2);
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                T v = ring[(slot * 2 + k) * RS + pos] + stage[k * NPIECE + t];
                if (hasy) { v += stage[k * NPIECE + NPX + r4 * RW + rx + 1]; v += stage[k * NPIECE + NPX + NPY + r4 * 4 + c4]; }
                ring[(slot * 2 + k) * RS + pos] = v;
            }
        } else {
            const int q = t - NPX, r4 = q / (RW - 4), rx = q % (RW - 4) + 1;
            const int ry = r4 == 0 ? -1 : (r4 == 1 ? 0 : (r4 == 2 ? TY - 1 : TY));
            const int pos = (ry + 1) * RW + rx + 1;
#pragma unroll
            for (int k = 0; k < 2; ++k) ring[(slot * 2 + k) * RS + pos] += stage[k * NPIECE + NPX + r4 * RW + rx + 1];
        }
    };

    // ---- pulls ------------------------------------------------------------------------------------
    // f_i(x) = h_i(x - c_i), or h_opp(i)(x) across a solid link
    auto src_of = [&](int k, int i, const long long (&zoff)[3], long long n, unsigned lk) -> const T* {
        if (HAS_SOLID && i > 0 && (lk >> dir_opp(i) & 1u)) return h + (long long)pop_plane(k, dir_opp(i)) * NP + n;
        return h + (long long)pop_plane(k, i) * NP + zoff[1 - dir_cz(i)] + ys[1 - dir_cy(i)] + xs[1 - dir_cx(i)];
    };
    auto plane_of = [&](int p, long long (&zoff)[3], long long& n, unsigned& lk) {
        zoff[0] = wrapz(p - 1) * pl; zoff[1] = wrapz(p) * pl; zoff[2] = wrapz(p + 1) * pl;
        n = zoff[1] + own_xy;
        lk = HAS_SOLID ? __ldg(links + n) : 0u;
    };
    auto prefetch_blue = [&](int p) {                          // -> stash, asynchronously
        long long zoff[3], n; unsigned lk;
        plane_of(p, zoff, n, lk);
        if (!HAS_SOLID || !(lk & OP_SOLID_BIT)) {
#pragma unroll
            for (int i = 0; i < Q; ++i) cp_async<sizeof(T)>(stash + i * NT + t, src_of(1, i, zoff, n, lk));
        }
        cp_async_commit();
    };
    auto prefetch_red = [&](int p, T (&fr)[Q]) {               // -> registers
        long long zoff[3], n; unsigned lk;
        plane_of(p, zoff, n, lk);
        if (!HAS_SOLID || !(lk & OP_SOLID_BIT)) {
#pragma unroll
            for (int i = 0; i < Q; ++i) fr[i] = __ldg(src_of(0, i, zoff, n, lk));
        }
    };

    // ---- prologue -----------------------------------------------------------------------------
    T fr[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) fr[i] = T(0);
    prefetch_red(z0 - 1, fr);
    __syncthreads();                                           // zero fill done before anything lands in `stage`
#pragma unroll 1
    for (int p = z0 - 2; p <= z0; ++p) {
        ring_issue(p);
        cp_async_wait<0>();
        __syncthreads();
        ring_assemble(p);
        __syncthreads();
    }
    prefetch_blue(z0 - 1);

    // z pipelines of this node's density partial sums: [k][0] = A_+1(z-1) + A_0(z) so far, [k][1] = A_+1(z)
    T own_acc[2][2] = {{T(0), T(0)}, {T(0), T(0)}};

    const T zero = T(0);
    auto from_left = [&](T v) { const T r = __shfl_up_sync(0xffffffffu, v, 1); return tx == 0 ? zero : r; };
    auto from_right = [&](T v) { const T r = __shfl_down_sync(0xffffffffu, v, 1); return tx == TX - 1 ? zero : r; };

#pragma unroll 1
    for (int z = z0 - 1; z <= z1; ++z) {
        const int zt = wrapz(z - 1), zl = wrapz(z);              // plane of the density target / of this plane
        const long long n = zl * pl + own_xy;
        const bool store_h = z >= z0 && z < z1;                 // planes z0-1 and z1 are re-collided only
        const bool store_rho = z - 1 >= z0;                     // target plane z-1 (always < z1 here)
        const bool more = z < z1;                               // iteration z+1 exists
        const int s0 = (z - z0 + 2) & 3;                        // ring slot of plane z
        unsigned lk = 0;
        if (HAS_SOLID) lk = __ldg(links + n);
        const bool fluid = !HAS_SOLID || !(lk & OP_SOLID_BIT);  // nothing happens inside a particle

        // x stage of the density gather for one opposite pair (h1 = direction 2p+1, h2 = 2p+2) of component k:
        // row sums into u0/up/um[cz+1], the tile's virtual columns -1 / TX into shared memory.
        auto xpair = [&](int k, int p, T h1, T h2, T (&u0)[3], T (&up)[3], T (&um)[3]) {
            T* sup0 = SU + (k * 6 + 1) * RS;                    // Up[dz = 0] plane
            T* sum0 = SU + (k * 6 + 4) * RS;                    // Um[dz = 0] plane
            T* e0k = e0a + k * 6 * TY;                          // [dz+1][side][TY]
            T l = zero, r = zero;
            if (p == 0 || (p >= 3 && p <= 6)) { l = from_left(h1); r = from_right(h2); }   // p is uniform: every lane shuffles
            if (p == 0) {                                       // +x / -x
                u0[1] += l; u0[1] += r;
                if (tx == TX - 1) e0k[(1 * 2 + 1) * TY + ty] = h1;
                if (tx == 0) e0k[(1 * 2 + 0) * TY + ty] = h2;
            } else if (p == 1) { up[1] = h1; um[1] = h2; }       // +y / -y
            else if (p == 2) { u0[2] = h1; u0[0] = h2; }         // +z / -z
            else if (p == 3) {                                  // +x+y / -x-y
                up[1] += l; um[1] += r;
                if (tx == TX - 1) sup0[own_r + 1] = h1;
                if (tx == 0) sum0[own_r - 1] = h2;
            } else if (p == 4) {                                // +x-y / -x+y
                um[1] += l; up[1] += r;
                if (tx == TX - 1) sum0[own_r + 1] = h1;
                if (tx == 0) sup0[own_r - 1] = h2;
            } else if (p == 5) {                                // +x+z / -x-z
                u0[2] += l; u0[0] += r;
                if (tx == TX - 1) e0k[(2 * 2 + 1) * TY + ty] = h1;
                if (tx == 0) e0k[(0 * 2 + 0) * TY + ty] = h2;
            } else if (p == 6) {                                // +x-z / -x+z
                u0[0] += l; u0[2] += r;
                if (tx == TX - 1) e0k[(0 * 2 + 1) * TY + ty] = h1;
                if (tx == 0) e0k[(2 * 2 + 0) * TY + ty] = h2;
            } else if (p == 7) { up[2] = h1; um[0] = h2; }       // +y+z / -y-z
            else { up[0] = h1; um[2] = h2; }                     // +y-z / -y+z
            // corner exports: only cz = 0 directions reach a diagonal tile, so target plane = this plane
            if (store_h && (p == 3 || p == 4)) {
                if (p == 3 && tx == TX - 1 && ty == TY - 1) ro.xy[k * ro.s_xy + zl * psxy + (btyp * ntx + btxp) * 4 + 0] = h1;
                if (p == 3 && tx == 0 && ty == 0) ro.xy[k * ro.s_xy + zl * psxy + (btym * ntx + btxm) * 4 + 3] = h2;
                if (p == 4 && tx == TX - 1 && ty == 0) ro.xy[k * ro.s_xy + zl * psxy + (btym * ntx + btxp) * 4 + 2] = h1;
                if (p == 4 && tx == 0 && ty == TY - 1) ro.xy[k * ro.s_xy + zl * psxy + (btyp * ntx + btxm) * 4 + 1] = h2;
            }
        };
        // publish the y-stage inputs of component k and export across the tile's y edges
        auto publish = [&](int k, const T (&up)[3], const T (&um)[3]) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                SU[(k * 6 + d) * RS + own_r] = up[d];
                SU[(k * 6 + 3 + d) * RS + own_r] = um[d];
            }
            if (ty == 0 || ty == TY - 1) {                      // the row beyond the edge receives exactly Um (Up)
                const int which = ty == 0 ? 0 : 1;
                T* acc = accr + ((k * 2 + which) * TX + tx) * 2;
                const T a_m = which == 0 ? um[0] : up[0], a_0 = which == 0 ? um[1] : up[1], a_p = which == 0 ? um[2] : up[2];
                const T out = acc[0] + a_m;
                acc[0] = acc[1] + a_0;
                acc[1] = a_p;
                if (store_rho) ro.y[k * ro.s_y + zt * psy + ((which == 0 ? btym : btyp) * 2 + (which == 0 ? 1 : 0)) * nx + x] = out;
            }
        };

        // ---- moments of both components, common velocity, force --------------------------------
        cp_async_wait<0>();                                      // this thread's stash slots have landed
        T rr = T(0), rb = T(0), ux = T(0), uy = T(0), uz = T(0);
        T er[3] = {T(0), T(0), T(0)}, eb[3] = {T(0), T(0), T(0)};
        if (fluid) {
            T jb[3] = {T(0), T(0), T(0)}, jr[3];
            rb = stash[t];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const T a = stash[(2 * p + 1) * NT + t], b = stash[(2 * p + 2) * NT + t];
                rb += a + b;
                const T d = a - b;
                if (pair_cx(p)) jb[0] += T(pair_cx(p)) * d;
                if (pair_cy(p)) jb[1] += T(pair_cy(p)) * d;
                if (pair_cz(p)) jb[2] += T(pair_cz(p)) * d;
            }
            // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6); a solid neighbour counts 0 (S7)
            T gr[3] = {T(0), T(0), T(0)}, gb[3] = {T(0), T(0), T(0)};
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                const int op = own_r + pair_cy(p) * RW + pair_cx(p), om = own_r - pair_cy(p) * RW - pair_cx(p);
                T bp = ring[(sp * 2 + 1) * RS + op], bm = ring[(sm_ * 2 + 1) * RS + om];
                T rp = ring[(sp * 2 + 0) * RS + op], rm = ring[(sm_ * 2 + 0) * RS + om];
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
            moments19<T>(fr, rr, jr[0], jr[1], jr[2]);
            const T den = om_r * rr + om_b * rb;                 // S4
            const T inv = den != T(0) ? T(1) / den : T(0);
            ux = (om_r * jr[0] + om_b * jb[0]) * inv;
            uy = (om_r * jr[1] + om_b * jb[1]) * inv;
            uz = (om_r * jr[2] + om_b * jb[2]) * inv;
            er[0] = ux - G * gr[0]; er[1] = uy - G * gr[1]; er[2] = uz - G * gr[2];
            eb[0] = ux - G * gb[0]; eb[1] = uy - G * gb[1]; eb[2] = uz - G * gb[2];
        }
        if (more) ring_issue(z + 2);                             // slot of plane z-2: last read one iteration ago

        // ---- blue: collide pair by pair out of the stash, store, x stage, publish -----------------
        T u0b[3] = {T(0), T(0), T(0)};
        {
            T up[3] = {T(0), T(0), T(0)}, um[3] = {T(0), T(0), T(0)};
            const T omc = T(1) - om_b;
            const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
            const T ae = T(1) - T(1.5) * (eb[0] * eb[0] + eb[1] * eb[1] + eb[2] * eb[2]);
            T* o = g + n;
            T bs = T(0);
            {
                const T h0 = fluid ? omc * stash[t] + w_rest<T>() * rb * (ae - omc * a0) : zero;
                if (fluid && store_h) o[(long long)pop_plane(1, 0) * NP] = h0;
                u0b[1] = h0;
            }
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                T h1 = zero, h2 = zero;
                if (fluid) {
                    const T cu = T(pair_cx(p)) * ux + T(pair_cy(p)) * uy + T(pair_cz(p)) * uz;
                    const T ce = T(pair_cx(p)) * eb[0] + T(pair_cy(p)) * eb[1] + T(pair_cz(p)) * eb[2];
                    const T wr = w_pair<T>(p) * rb;
                    const T sym = wr * ((ae + T(4.5) * ce * ce) - omc * (a0 + T(4.5) * cu * cu));
                    const T asym = (T(3) * wr) * (ce - omc * cu);
                    h1 = omc * stash[(2 * p + 1) * NT + t] + (sym + asym);
                    h2 = omc * stash[(2 * p + 2) * NT + t] + (sym - asym);
                    if (store_h) { o[(long long)pop_plane(1, 2 * p + 1) * NP] = h1; o[(long long)pop_plane(1, 2 * p + 2) * NP] = h2; }
                    if (HAS_SOLID) {                             // bounced-back arrivals of the next step come from this node
                        if (lk >> (2 * p + 1) & 1u) bs += h1;
                        if (lk >> (2 * p + 2) & 1u) bs += h2;
                    }
                }
                xpair(1, p, h1, h2, u0b, up, um);
            }
            if (HAS_SOLID) u0b[1] += bs;
            publish(1, up, um);
        }
        if (more) prefetch_blue(z + 1);

        // ---- red: collide out of the registers, store, x stage, publish ---------------------------
        T u0r[3] = {T(0), T(0), T(0)};
        {
            T up[3] = {T(0), T(0), T(0)}, um[3] = {T(0), T(0), T(0)};
            T bs = T(0);
            if (fluid) {
                collide19<T>(fr, rr, T(1) - om_r, ux, uy, uz, er[0], er[1], er[2]);
                if (store_h) {
#pragma unroll
                    for (int i = 0; i < Q; ++i) g[(long long)pop_plane(0, i) * NP + n] = fr[i];
                }
                if (HAS_SOLID) {
#pragma unroll
                    for (int i = 1; i < Q; ++i)
                        if (lk >> i & 1u) bs += fr[i];
                }
            }
            u0r[1] = fluid ? fr[0] : zero;
#pragma unroll
            for (int p = 0; p < 9; ++p) xpair(0, p, fluid ? fr[2 * p + 1] : zero, fluid ? fr[2 * p + 2] : zero, u0r, up, um);
            if (HAS_SOLID) u0r[1] += bs;
            publish(0, up, um);
        }
        if (more) {
            prefetch_red(z + 1, fr);
            cp_async_wait<1>();                                  // the ring pieces of plane z+2 (the stash may still fly)
        }
        __syncthreads();

        // ---- y stage and z pipeline of the gather; exports across the tile's x edges ---------------
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const T* u0 = k == 0 ? u0r : u0b;
            T a[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                a[d] = u0[d] + SU[(k * 6 + d) * RS + own_r - RW];          // Up[dz](y-1)
                a[d] += SU[(k * 6 + 3 + d) * RS + own_r + RW];             // Um[dz](y+1)
            }
            const T out = own_acc[k][0] + a[0];
            own_acc[k][0] = own_acc[k][1] + a[1];
            own_acc[k][1] = a[2];
            if (store_rho) ro.in[k * ro.s_in + (long long)zt * pl + own_xy] = out;
            if (tx == 0 || tx == TX - 1) {
                const int side = tx == 0 ? 0 : 1;
                const int vc = tx == 0 ? own_r - 1 : own_r + 1;            // the virtual column next to this lane
                const T* e0k = e0a + k * 6 * TY;
                T a_0 = e0k[(1 * 2 + side) * TY + ty] + SU[(k * 6 + 1) * RS + vc - RW];
                a_0 += SU[(k * 6 + 4) * RS + vc + RW];
                const T a_m = e0k[(0 * 2 + side) * TY + ty], a_p = e0k[(2 * 2 + side) * TY + ty];
                T* acc = accc + ((k * 2 + side) * TY + ty) * 2;
                const T hout = acc[0] + a_m;
                acc[0] = acc[1] + a_0;
                acc[1] = a_p;
                if (store_rho) ro.x[k * ro.s_x + zt * psx + ((bty * ntx + (side == 0 ? btxm : btxp)) * 2 + (side == 0 ? 1 : 0)) * TY + ty] = hout;
            }
        }
        if (more) ring_assemble(z + 2);
        __syncthreads();
    }
}

}  // namespace lb
