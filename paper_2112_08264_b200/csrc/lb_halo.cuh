// lb_halo.cuh -- the fused one-pass time step for boxes without solid nodes: the hot kernel on B200.
//
// Same algorithm, state convention (h-state, pull streaming) and warp-specialised structure as lb_tma.cuh, with the two
// sources of wasted DRAM traffic of that kernel removed (measured there: 685-697 B/node against 608 algorithmic):
//
//   * x shift without wide boxes.  A TMA box must start 16-byte aligned, so lb_tma.cuh pulls the directions with
//     c_x != 0 as boxes 16 bytes wider than the tile: 9 sectors per row instead of 8, and the ninth misses in L2
//     (-5 % with the margins switched off).  Here EVERY box is the aligned 32 x TY tile, and the one column a tile needs
//     from its x neighbour comes from a small second copy the neighbour writes for it, the x-halo arrays
//         hx[2 j + k][z][tile_x][y'] = h_i(column, (y' - c_iy) mod ny, z),    i = the j-th direction with c_x != 0,
//     column = the tile's last column for c_x > 0, its first for c_x < 0.  The writer stores its value at row y + c_iy
//     (mod ny): the reader's box is then rows y0 .. y0 + TY - 1 for every direction -- 16-byte aligned, never out of
//     range in y, and periodic in x through the tile index.  5 B/node written + 5 read instead of ~20 read.
//   * density without a carried full field.  lb_tma.cuh carries rho(t+1) of every node from step to step (16 B/node
//     written, ~24 read).  Here the staged populations of plane z+1 are summed once more (19 LDS + 18 adds per thread)
//     one iteration before that plane is collided: rho^k(x, t) = sum_i h_i(x - c_i) for the tile's own nodes goes
//     straight into the shared-memory density ring.  Only the one-node FRAME around the tile still comes from carried
//     single-writer arrays: the owner tile's gather over its own post-collision values for its edge rows / columns
//     (er, ec) plus what its x / y / diagonal neighbours exported (x, y, xy), added in the fixed order
//     ((in + x) + y) + xy by three ring warps.  ~10 B/node instead of ~45.
//     Two more planes are staged per z chunk (z0-2 and z0+zc+1, summed only).
//
// Per-step diagnostics (DIAG): mass per component and total momentum of the state AFTER this step, accumulated per
// thread in shared memory (double), reduced by warp shuffles and written as one partial per CTA; k_diag_final adds the
// partials in a fixed order.
#pragma once
#include <cuda.h>

#include "lb_lattice.cuh"
#include "lb_tma.cuh"

namespace lb {

// the carried single-writer arrays of the frame density (both components each)
template <typename T>
struct EdgeView {
    T* er;                      // [k][z][tile_y][side][nx]            own gather, rows y_local = 0 (side 0) and TY-1 (side 1)     (stride s_y)
    T* ec;                      // [k][z][tile_y][tile_x][side][TY]    own gather, columns x_local = 0 and TX-1                    (stride s_x)
    T* x;  long long s_x;       // [k][z][tile_y][tile_x][side][TY]    what the x neighbour sent to those columns
    T* y;  long long s_y;       // [k][z][tile_y][side][nx]            what the y neighbour sent to those rows
    T* xy; long long s_xy;      // [k][z][tile_y][tile_x][4]           what the diagonal neighbours sent to the corners
};

// j-th direction with c_x != 0: directions 1, 2, 7 .. 14 -> j = 0 .. 9
__host__ __device__ constexpr int halo_j(int i) { return i <= 2 ? i - 1 : i - 5; }
constexpr int NHALO = 10;

template <typename T, int TY>
struct HaloLayout {
    static constexpr int TX = 32, NT = TX * TY;
    static constexpr int RW = TX + 2, RH = TY + 2, RS = RW * RH;       // density ring plane: tile + one-node frame
    static constexpr int SUP = TY * RW;                                // one y-stage plane: tile rows with an x frame
    static constexpr int NFRAME = 2 * RW + 2 * TY;                     // frame positions of a ring plane
    // one stage slot per direction, both components in it: [k][TY][TX]; slots of the directions with c_x != 0 are followed
    // by the x-halo box [k][TY], padded to 128 bytes.  TMA destinations are 128-byte aligned.
    static constexpr int NA = 2 * NT;
    static constexpr int HXE = 128 / int(sizeof(T));
    static constexpr int WA = NA + HXE;
    static_assert(2 * TY <= HXE && (NA * sizeof(T)) % 128 == 0, "TMA destination alignment");
    __host__ __device__ static constexpr int wide_before(int i) { return (i > 1) + (i > 2) + (i > 7 ? (i - 7 < 8 ? i - 7 : 8) : 0); }
    __host__ __device__ static constexpr int slot_off(int i) { return (i - wide_before(i)) * NA + wide_before(i) * WA; }
    static constexpr int STAGE_ELEMS = slot_off(Q);
    static constexpr unsigned STAGE_TX_BYTES = unsigned((Q * NA + NHALO * 2 * TY) * sizeof(T));
    static constexpr int STAGE = 0;                                    // [2][STAGE_ELEMS]
    static constexpr int RING = STAGE + 2 * STAGE_ELEMS;               // [4][2][RS]      rho(t), planes z-1..z+2
    static constexpr int SU = RING + 8 * RS;                           // [2][2][2][SUP]  double-buffered z-summed Up, Um per component
    static constexpr int LAND = SU + 8 * SUP;                          // [2][4][96]      landing slots of the frame pieces, per component and ring thread
    static constexpr int EXR = 24;                                     // one record per (component, tile row, x side): [0..4] the density export
                                                                       // state, [8 + 5 b + m] the x-halo copy of pair m (c_x != 0) of an iteration with parity b
    static constexpr int EX = LAND + 2 * 4 * 96;                       // [2 TY][2][EXR]
    static constexpr int CST = EX + 2 * TY * 2 * EXR;                  // {om_r, om_b, G}
    static constexpr int END = CST + 4;
    static constexpr size_t DIAG_BYTE_OFF = (size_t(END) * sizeof(T) + 15) / 16 * 16;      // double [4][2 NT] (DIAG only)
    static constexpr size_t DIAG_BYTES = size_t(4) * 2 * NT * sizeof(double);
    template <bool DIAG> __host__ __device__ static constexpr size_t bar_byte_off() { return DIAG_BYTE_OFF + (DIAG ? DIAG_BYTES : 0); }
    static constexpr int NBARS = 5 + 8 * TY;                           // full[2], done[2], rdy, rowpub[2][2 TY], rhopub[2][2 TY]
    template <bool DIAG> __host__ __device__ static constexpr size_t bytes() { return bar_byte_off<DIAG>() + NBARS * sizeof(unsigned long long); }
    static_assert(DIAG_BYTE_OFF + DIAG_BYTES + NBARS * 8 <= 227 * 1024, "shared memory per CTA");
};

// Slow paths of the one warp of a y-boundary tile whose row pulls from beyond the box edge (the TMA zero-fills there; periodic,
// PAPER.md:160): out of line, so that the other warps do not carry their address arithmetic as predicated-off instructions.
template <typename T>
__device__ __noinline__ T ywrap_load(const T* __restrict__ h, long long NP, int nx, int ny, int nz, int k, int i, int x, int gy, int z) {
    const int cx = dir_cx(i), cz = dir_cz(i);
    const int xs = cx > 0 ? (x == 0 ? nx - 1 : x - 1) : (cx < 0 ? (x == nx - 1 ? 0 : x + 1) : x);
    const int zz = cz > 0 ? (z == 0 ? nz - 1 : z - 1) : (cz < 0 ? (z + 1 == nz ? 0 : z + 1) : z);
    return __ldg(h + (long long)pop_plane(k, i) * NP + ((long long)zz * ny + gy) * nx + xs);
}
template <typename T, typename L>
__device__ __noinline__ T plane_density_ywrap(const T* st, int rd0, int rdp, int rdm, bool ylo, const T* __restrict__ h, long long NP,
                                              int nx, int ny, int nz, int k, int x, int z) {
    const int gy = ylo ? ny - 1 : 0;
    auto get = [&](int i) -> T {
        const int cy = dir_cy(i), cx = dir_cx(i);
        if ((cy > 0 && ylo) || (cy < 0 && !ylo)) return ywrap_load<T>(h, NP, nx, ny, nz, k, i, x, gy, z);
        return st[L::slot_off(i) + (cx == 0 ? rd0 : (cx > 0 ? rdp : rdm))];
    };
    T r = get(0);
#pragma unroll 1
    for (int p = 0; p < 9; ++p) r += get(2 * p + 1) + get(2 * p + 2);
    return r;
}

// Threads: 2 NT consumers (component k = t / NT, node (tx, ty): one warp per tile row and component) + one producer warp
// group (TMA warp + 3 ring warps) that hands its registers to the consumers.
template <typename T, bool DIAG, int TY>
__global__ void __launch_bounds__(2 * 32 * TY + 128, 1)
k_step_halo(const __grid_constant__ CUtensorMap tm_n, const __grid_constant__ CUtensorMap tm_h,
            const T* __restrict__ h, T* __restrict__ g, T* __restrict__ hxo, const EdgeView<T> ri, const EdgeView<T> ro,
            double* __restrict__ diag_part, long long NP, int nx, int ny, int nz, int zc, T om_r, T om_b, T G) {
    using L = HaloLayout<T, TY>;
    constexpr int TX = L::TX, NT = L::NT, NC = 2 * NT, RW = L::RW, RS = L::RS, SUP = L::SUP;
    static_assert(TY >= 2 && TY <= 8, "one named barrier per tile row (ids 1..TY)");
    constexpr int START_REGS = (65536 / (NC + 128)) / 8 * 8;
    constexpr int PRODUCER_REGS = 32;
    constexpr int CONSUMER_REGS = (START_REGS + (START_REGS - PRODUCER_REGS) * 128 / NC) / 8 * 8;
    extern __shared__ __align__(1024) unsigned char smem_halo[];
    T* sm = reinterpret_cast<T*>(smem_halo);
    T* stage = sm + L::STAGE;
    T* ring = sm + L::RING;
    T* SUb = sm + L::SU;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_halo + L::template bar_byte_off<DIAG>());
    unsigned long long* full = bars;          // [2] the boxes of staged plane j have landed in stage j & 1 (tx bytes)
    unsigned long long* done = bars + 2;      // [2] every consumer warp has taken what it needs out of stage j & 1
    unsigned long long* rdy = bars + 4;       // the ring warps have put the frame of the density ring plane this iteration adds in place
    unsigned long long* rowpub = bars + 5;    // [2][2 TY] warp (k, ty) has published its y-stage inputs of this plane
    unsigned long long* rhopub = bars + 5 + 4 * TY;   // [2][2 TY] warp (k, ty) has put rho^k of its row of the next plane into the ring

    const int t = threadIdx.x;
    const int ntx = nx / TX, nty = ny / TY;
    const int btx = blockIdx.x, bty = blockIdx.y;
    const int x0 = btx * TX, y0 = bty * TY;
    const int z0 = blockIdx.z * zc;           // the host guarantees nz % zc == 0
    const int niter = zc + 2;                 // collided planes z0-1 .. z0+zc; the first and the last are re-collided only
    const int nstaged = zc + 4;               // staged planes p_j = z0-2+j: the outermost two are summed only (density)
    const long long pl = (long long)nx * ny;
    const int btxm = btx == 0 ? ntx - 1 : btx - 1, btxp = btx == ntx - 1 ? 0 : btx + 1;
    const int btym = bty == 0 ? nty - 1 : bty - 1, btyp = bty == nty - 1 ? 0 : bty + 1;
    auto wrapz = [&](int p) { p %= nz; return p < 0 ? p + nz : p; };

    if (t == 0) {
        for (int s = 0; s < 2; ++s) { mbar_init(full + s, 1); mbar_init(done + s, 2 * TY); }
        mbar_init(rdy, 3);
        for (int b = 0; b < 8 * TY; ++b) mbar_init(rowpub + b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        sm[L::CST + 0] = om_r; sm[L::CST + 1] = om_b; sm[L::CST + 2] = G;
    }
    __syncthreads();

    // =================================== producer warp group ===================================
    if (t >= NC) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
        if (t >= NC + 32) {
            // ---- ring warps (3): the FRAME of the density ring, one plane per iteration.  Thread r < NFRAME owns one frame
            //      position of both components: its value is ((in + x) + y) + xy of up to four single-writer pieces (header),
            //      fetched with cp.async one iteration ahead into landing slots only this thread reads. ----
            const int r = t - NC - 32;
            int oin = -1, ox = -1, oy = -1, oxy = -1, pos = 0;
            bool in_row = false;
            if (r < L::NFRAME) {
                int rx, ry;
                if (r < RW) { rx = r - 1; ry = -1; }
                else if (r < 2 * RW) { rx = r - RW - 1; ry = TY; }
                else if (r < 2 * RW + TY) { rx = -1; ry = r - 2 * RW; }
                else { rx = TX; ry = r - 2 * RW - TY; }
                pos = (ry + 1) * RW + rx + 1;
                const int otx = rx < 0 ? btxm : (rx >= TX ? btxp : btx), oty = ry < 0 ? btym : (ry >= TY ? btyp : bty);
                const int lx = rx < 0 ? TX - 1 : (rx >= TX ? 0 : rx), ly = ry < 0 ? TY - 1 : (ry >= TY ? 0 : ry);
                const bool xe = lx == 0 || lx == TX - 1, ye = ly == 0 || ly == TY - 1;   // edge column / row of its owner tile
                const int o_row = (oty * 2 + (ly != 0)) * nx + otx * TX + lx;           // er / y entry of an edge-row node
                const int o_col = ((oty * ntx + otx) * 2 + (lx != 0)) * TY + ly;        // ec / x entry of an edge-column node
                in_row = ye;
                oin = ye ? o_row : o_col;
                if (xe) ox = o_col;
                if (ye) oy = o_row;
                if (xe && ye) oxy = (oty * ntx + otx) * 4 + (ly != 0) * 2 + (lx != 0);
            }
            const unsigned psx_ = unsigned(nty * ntx * 2 * TY), psy_ = unsigned(nty * 2 * nx), psxy_ = unsigned(nty * ntx * 4);
            T* land = sm + L::LAND + r;                                    // [2][4][96]
            auto frame_fetch = [&](int j) {                                // pieces of staged plane j
                if (oin >= 0) {
                    const unsigned zp = unsigned(wrapz(z0 - 2 + j));
                    const T* s_in = in_row ? ri.er + (zp * psy_ + unsigned(oin)) : ri.ec + (zp * psx_ + unsigned(oin));
                    const long long cs_in = in_row ? ri.s_y : ri.s_x;
                    cp_async<sizeof(T)>(land, s_in);
                    cp_async<sizeof(T)>(land + 4 * 96, s_in + cs_in);
                    if (ox >= 0) {
                        const T* s = ri.x + (zp * psx_ + unsigned(ox));
                        cp_async<sizeof(T)>(land + 96, s);
                        cp_async<sizeof(T)>(land + 5 * 96, s + ri.s_x);
                    }
                    if (oy >= 0) {
                        const T* s = ri.y + (zp * psy_ + unsigned(oy));
                        cp_async<sizeof(T)>(land + 2 * 96, s);
                        cp_async<sizeof(T)>(land + 6 * 96, s + ri.s_y);
                    }
                    if (oxy >= 0) {
                        const T* s = ri.xy + (zp * psxy_ + unsigned(oxy));
                        cp_async<sizeof(T)>(land + 3 * 96, s);
                        cp_async<sizeof(T)>(land + 7 * 96, s + ri.s_xy);
                    }
                }
                cp_async_commit();
            };
            auto frame_assemble = [&](int j) {
                cp_async_wait<0>();
                if (oin >= 0) {
                    T* dst = ring + (j & 3) * 2 * RS + pos;
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {
                        const T* ld = land + kk * 4 * 96;
                        T v = ld[0];
                        if (ox >= 0) v += ld[96];
                        if (oy >= 0) v += ld[2 * 96];
                        if (oxy >= 0) v += ld[3 * 96];
                        dst[kk * RS] = v;
                    }
                }
            };
            // x-halo copies (header): thread r < 8 NHALO writes, for both components, the value of the r / TY-th direction with
            // c_x != 0 that the edge lane of tile row r % TY left in its export record, at row y + c_iy (periodic)
            const int hj = r / TY, hrow = r % TY;
            const int hi_ = hj < 2 ? hj + 1 : hj + 5;                      // that direction
            unsigned eh0 = 0;
            const T* hrec = sm + L::EX + (hrow * 2 + (hj & 1 ? 0 : 1)) * L::EXR + 8 + hj / 2;   // odd directions (c_x > 0) come from lane_hi
            if (r < TY * NHALO) {
                int yy = y0 + hrow + dir_cy(hi_);
                yy = yy < 0 ? yy + ny : (yy >= ny ? yy - ny : yy);
                eh0 = (unsigned(2 * hj) * unsigned(nz) * unsigned(ntx) + unsigned(btx)) * unsigned(ny) + unsigned(yy);
            }
            const unsigned hk = unsigned(nz) * unsigned(ntx) * unsigned(ny);   // component stride
            auto halo_out = [&](int it) {                                  // the copies of collided plane z0 - 1 + it
                if (r < TY * NHALO) {
                    const unsigned ph_ = (it >> 1) & 1;
                    mbar_wait(rowpub + (it & 1) * 2 * TY + hrow, ph_);      // both warps of that tile row are past their collision
                    mbar_wait(rowpub + (it & 1) * 2 * TY + TY + hrow, ph_);
                    const unsigned e = eh0 + unsigned(wrapz(z0 - 1 + it)) * unsigned(ntx * ny);
                    const T* rec = hrec + (it & 1) * 5;
                    hxo[e] = rec[0];
                    hxo[e + hk] = rec[TY * 2 * L::EXR];
                }
            };
            for (int j = 0; j < 2; ++j) {                                  // iteration 0 needs ring planes 0, 1, 2
                frame_fetch(j);
                frame_assemble(j);
            }
            frame_fetch(2);
            for (int it = 0; it < niter; ++it) {
                // ring plane it+2: its slot held plane it-2, last read in iteration it-2, which every consumer warp had left
                // when it arrived on done for staged plane `it` (in iteration it-1)
                // (from it = 1 on, so that no ring warp arrives on rdy for iteration it before all three have arrived for it - 1:
                // a consumer warp arrives on done after it has waited for rdy)
                if (it >= 1) mbar_wait(done + (it & 1), (it >> 1) & 1);
                frame_assemble(it + 2);
                __syncwarp();
                if ((r & 31) == 0) mbar_arrive(rdy);
                if (it + 3 < nstaged) frame_fetch(it + 3);
                // the consumers overwrite the records of iteration it - 1 in iteration it + 1, for which they need this warp's next
                // arrival on rdy: program order keeps the copies safe
                if (it >= 1) halo_out(it - 1);
            }
            halo_out(niter - 1);
            return;
        }
        // ---- TMA warp: staged plane j goes into stage j & 1 as soon as every consumer warp has left plane j - 2 ----
        const int lane = t - NC;
        const unsigned long long pol = l2_policy_evict_normal();    // no box is read twice here
        for (int j = 0; j < nstaged; ++j) {
            const int z = z0 - 2 + j;
            const int zw[3] = {wrapz(z - 1), wrapz(z), wrapz(z + 1)};
            if (lane == 0) {
                const int s = j & 1;
                if (j >= 2) mbar_wait(done + s, ((j >> 1) - 1) & 1);
                mbar_expect_tx(full + s, L::STAGE_TX_BYTES);
#pragma unroll
                for (int i = 0; i < Q; ++i) {
                    const int zq = zw[1 - dir_cz(i)];                       // f_i(x) = h_i(x - c_i)
                    T* slot = stage + s * L::STAGE_ELEMS + L::slot_off(i);
                    tma_load_4d(slot, &tm_n, full + s, x0, y0 - dir_cy(i), zq, pop_plane(0, i), pol);   // planes q, q + 1: both components
                    if (dir_cx(i) != 0)                                     // the neighbour's column, rows pre-shifted by the writer
                        tma_load_4d(slot + L::NA, &tm_h, full + s, y0, dir_cx(i) > 0 ? btxm : btxp, zq, 2 * halo_j(i), pol);
                }
            }
            __syncwarp();
        }
        return;
    }

    // =================================== consumers ===================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
    const int k = t / NT;                                                  // component of this thread (warp-uniform)
    const int tl = t - k * NT;
    const int tx = tl % TX, ty = tl / TX;
    const bool lane_lo = tx == 0, lane_hi = tx == TX - 1, row_lo = ty == 0, row_hi = ty == TY - 1;
    const int own_r = (ty + 1) * RW + tx + 1;
    const T zero = T(0);
    const T omc = T(1) - (k == 0 ? om_r : om_b);
    const unsigned e_own = unsigned((long long)k * NP + (long long)(y0 + ty) * nx + x0 + tx);
    auto opaque = [](int v) { asm volatile("" : "+r"(v)); return v; };
    const unsigned psx = unsigned(nty * ntx * 2 * TY), psy = unsigned(nty * 2 * nx), psxy = unsigned(nty * ntx * 4), plu = unsigned(pl);
    const unsigned step16 = unsigned((2 * NP * (long long)sizeof(T)) >> 4);
    const T* ring_o = ring + (1 - k) * RS + own_r;                         // the OTHER component's density (S2), at this node
    T* ring_w = ring + k * RS + own_r;                                     // where this thread puts rho^k of its node
    T* SUk = SUb + k * 2 * SUP + own_r - RW;
    T* exs = sm + L::EX + ((k * TY + ty) * 2 + (lane_hi ? 1 : 0)) * L::EXR;
    const volatile T* cst = sm + L::CST;
    // where this thread finds f_i = h_i(x - c_i) inside slot i, by c_x; the lane at the tile edge reads the x-halo box
    const int rd0 = k * NT + ty * TX + tx;
    const int rdp = lane_lo ? L::NA + k * TY + ty : rd0 - 1;
    const int rdm = lane_hi ? L::NA + k * TY + ty : rd0 + 1;
    const bool wrap_ylo = bty == 0 && row_lo, wrap_yhi = bty == nty - 1 && row_hi;   // warp-uniform: the TMA zero-fills rows outside the box
    if (lane_lo || lane_hi) { exs[3] = zero; exs[4] = zero; }
    double* dacc = reinterpret_cast<double*>(smem_halo + L::DIAG_BYTE_OFF) + t;      // [4][NC]: rho, and the post-collision momentum
    if (DIAG) { dacc[0] = 0.0; dacc[NC] = 0.0; dacc[2 * NC] = 0.0; dacc[3 * NC] = 0.0; }

    // rho^k of this node in a staged plane (Eq. 6), summed in the order of moments19
    auto plane_density = [&](const T* stp, int zp) -> T {
        if (wrap_ylo || wrap_yhi) return plane_density_ywrap<T, L>(stp, rd0, rdp, rdm, wrap_ylo, h, NP, nx, ny, nz, k, x0 + tx, zp);
        T r = stp[L::slot_off(0) + rd0];
#pragma unroll
        for (int p = 0; p < 9; ++p) {
            const int i1 = 2 * p + 1, i2 = 2 * p + 2;
            r += stp[L::slot_off(i1) + (dir_cx(i1) == 0 ? rd0 : (dir_cx(i1) > 0 ? rdp : rdm))]
               + stp[L::slot_off(i2) + (dir_cx(i2) == 0 ? rd0 : (dir_cx(i2) > 0 ? rdp : rdm))];
        }
        return r;
    };

    // ---- prologue: density of staged planes 0 and 1 ----
    mbar_wait(full + 0, 0);
    ring_w[0] = plane_density(stage, wrapz(z0 - 2));
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (lane_lo) mbar_arrive(done + 0);                                    // staged plane 0 is only summed
    mbar_wait(full + 1, 0);
    ring_w[2 * RS] = plane_density(stage + L::STAGE_ELEMS, wrapz(z0 - 1));

    T qa0 = zero, qb0 = zero, qap = zero, qbp = zero, qam = zero, qbm = zero;   // z pipelines of the density gather
    int zl = wrapz(z0 - 1), zt = wrapz(z0 - 2);         // this plane / the plane the gathered density belongs to

#pragma unroll 1
    for (int it = 0; it < niter; ++it) {
        const bool store_h = it >= 1 && it <= niter - 2;
        const bool store_rho = it >= 2;                 // target plane z-1 lies in [z0, z1)
        const int s0 = (it + 1) & 3;                    // ring slot of this plane (staged plane it + 1)
        const int sg = it & 1;                          // y-stage / rowpub buffer of this iteration
        const unsigned ph = (it >> 1) & 1;
        T* st = stage + ((it + 1) & 1) * L::STAGE_ELEMS;
        T* SU = SUk + sg * 4 * SUP;

        mbar_wait(rdy, it & 1);                         // the frame of ring planes z-1, z, z+1 is in place (the ring warps run ahead)

        // ---- pull: the stage holds h_i(x - c_i) for the whole tile (Eq. 5, periodic); it landed before last iteration's sum ----
        T f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = st[L::slot_off(i) + (dir_cx(i) == 0 ? rd0 : (dir_cx(i) > 0 ? rdp : rdm))];
        if (wrap_ylo || wrap_yhi) {
            const int gy = wrap_ylo ? ny - 1 : 0;
#pragma unroll
            for (int i = 1; i < Q; ++i)
                if (dir_cy(i) != 0) {
                    if ((dir_cy(i) > 0) == wrap_ylo) f[i] = ywrap_load<T>(h, NP, nx, ny, nz, k, i, x0 + tx, gy, zl);
                }
        }

        // ---- moments of this component (Eq. 6-7), exchanged with the other component's thread of the same node through
        //      stage entries this thread has just consumed ----
        T rho, jx, jy, jz;
        moments19<T>(f, rho, jx, jy, jz);
        {
            T* mine = st + rd0;
            mine[L::slot_off(0)] = rho; mine[L::slot_off(3)] = jx; mine[L::slot_off(4)] = jy; mine[L::slot_off(5)] = jz;
        }
        asm volatile("bar.sync %0, 64;" ::"r"(ty + 1) : "memory");         // the two warps (red, blue) of this tile row
        T ux, uy, uz;
        {
            const T* other = st + rd0 + (1 - 2 * k) * NT;
            const T orho = other[L::slot_off(0)], ojx = other[L::slot_off(3)], ojy = other[L::slot_off(4)], ojz = other[L::slot_off(5)];
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy accesses to the stage before the TMA's next writes
            __syncwarp();
            if (lane_lo) mbar_arrive(done + ((it + 1) & 1));               // the producer may refill this stage with staged plane it + 3
            // common velocity (S4); both threads of the node must get the same bits: commutative arithmetic only
            const T om_own = cst[k], om_oth = cst[1 - k];
            const T den = add_rn(mul_rn(om_own, rho), mul_rn(om_oth, orho));
            const T inv = den != zero ? T(1) / den : zero;
            ux = add_rn(mul_rn(om_own, jx), mul_rn(om_oth, ojx)) * inv;
            uy = add_rn(mul_rn(om_own, jy), mul_rn(om_oth, ojy)) * inv;
            uz = add_rn(mul_rn(om_own, jz), mul_rn(om_oth, ojz)) * inv;
        }

        // ---- density of the NEXT plane's own nodes into the ring (staged plane it + 2, stage it & 1).  With two stages, the earlier
        //      this sum the shorter the time that stage has to land, and a stage takes about one iteration to land when the kernel
        //      runs at the DRAM rate: measured, summing right after the pull costs 10 %, at the top of the iteration 18 % ----
        mbar_wait(full + (it & 1), ((it + 2) >> 1) & 1);
        ring_w[((it + 2) & 3) * 2 * RS] = plane_density(stage + (it & 1) * L::STAGE_ELEMS, zl + 1 == nz ? 0 : zl + 1);
        __syncwarp();
        if (lane_lo) mbar_arrive(rhopub + sg * 2 * TY + k * TY + ty);
        {   // the force needs the OTHER component's density in the rows y-1, y, y+1 of that plane
            unsigned long long* ob = rhopub + sg * 2 * TY + (1 - k) * TY + ty;
            if (row_lo) mbar_wait2(ob, ob + 1, ph);
            else if (row_hi) mbar_wait2(ob - 1, ob, ph);
            else mbar_wait3(ob - 1, ob, ob + 1, ph);
        }

        T ex, ey, ez;
        {
            // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6)
            T d[9];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                const T vp = ring_o[sp * 2 * RS + pair_cy(p) * RW + pair_cx(p)];
                const T vm = ring_o[sm_ * 2 * RS - pair_cy(p) * RW - pair_cx(p)];
                d[p] = w_pair<T>(p) * (vp - vm);
            }
            const T gx = (((d[0] + d[3]) + d[4]) + d[5]) + d[6];
            const T gy = (((d[1] + d[3]) - d[4]) + d[7]) + d[8];
            const T gz = (((d[2] + d[5]) - d[6]) + d[7]) - d[8];
            const T G_ = cst[2];
            ex = ux - G_ * gx; ey = uy - G_ * gy; ez = uz - G_ * gz;
        }
        if (DIAG && store_h) {
            // mass and momentum of the state after this step: streaming in a periodic box permutes the post-collision values, and
            // their moments are sum_i f*_i = rho, sum_i f*_i c_i = (1 - om) j + om rho u' + rho du (Eq. 1, Eq. 10, S5)
            const double om = 1.0 - double(omc), r_ = double(rho);
            dacc[0] += r_;
            dacc[NC] += double(omc) * double(jx) + r_ * (om * double(ux) + (double(ex) - double(ux)));
            dacc[2 * NC] += double(omc) * double(jy) + r_ * (om * double(uy) + (double(ey) - double(uy)));
            dacc[3 * NC] += double(omc) * double(jz) + r_ * (om * double(uz) + (double(ez) - double(uz)));
        }

        // ---- BGK collision with exact-difference forcing (Eq. 1, Eq. 10, S5), and, pair by pair as the post-collision values
        //      appear: their (aligned, coalesced) stores, the x-halo copies, and the x stage of the density gather
        //      rho(y, t+1) = sum_i h_i(y - c_i) for the tile's edge nodes and its neighbours' (lb_tma.cuh) ----
        T qc0 = zero, qcp = zero, qcm = zero;
        T* SUup = SU;
        T* SUum = SU + SUP;
        // every plane is stored, also the two re-collided ones at the chunk ends: their owner chunk writes the same bits
        T* o = g + (e_own + zl * plu);
        auto put = [&](T v) {
            st_global(o, v);
            ptr_step16(o, step16);
        };
        // x-halo copies: the edge lanes leave their values of the 5 pairs with c_x != 0 (lane_hi: the odd member, lane_lo: the even one)
        // in their export record; the ring warps write them out (header)
        T* exh = exs + 8 + sg * 5;
        collide19_pairs<T>(f, rho, omc, ux, uy, uz, ex, ey, ez,
            [&](T h0) { put(h0); qb0 += h0; },
            [&](int p, T h1, T h2) {
                put(h1);
                put(h2);
                T l = zero, r = zero;
                if (p == 0 || (p >= 3 && p <= 6)) {
                    l = __shfl_up_sync(0xffffffffu, h1, 1); r = __shfl_down_sync(0xffffffffu, h2, 1);
                    if (lane_lo || lane_hi) exh[p == 0 ? 0 : p - 2] = lane_hi ? h1 : h2;
                }
                if (p == 0) {                                              // +x / -x
                    if (!lane_lo) qb0 += l;
                    if (!lane_hi) qb0 += r;
                    if (lane_hi) exs[1] = h1;
                    if (lane_lo) exs[1] = h2;
                } else if (p == 1) { qbp += h1; qbm += h2; }                  // +y / -y
                else if (p == 2) { qc0 = h1; qa0 += h2; }                     // +z / -z
                else if (p == 3) {                                         // +x+y / -x-y
                    qbp += lane_lo ? zero : l;
                    qbm += lane_hi ? zero : r;
                    if (lane_hi) SUup[1] = h1;
                    if (lane_lo) SUum[-1] = h2;
                } else if (p == 4) {                                       // +x-y / -x+y
                    qbm += lane_lo ? zero : l;
                    qbp += lane_hi ? zero : r;
                    if (lane_hi) SUum[1] = h1;
                    if (lane_lo) SUup[-1] = h2;
                } else if (p == 5) {                                       // +x+z / -x-z
                    if (!lane_lo) qc0 += l;
                    if (!lane_hi) qa0 += r;
                    if (lane_hi) exs[2] = h1;
                    if (lane_lo) exs[0] = h2;
                } else if (p == 6) {                                       // +x-z / -x+z
                    if (!lane_lo) qa0 += l;
                    if (!lane_hi) qc0 += r;
                    if (lane_hi) exs[0] = h1;
                    if (lane_lo) exs[2] = h2;
                } else if (p == 7) { qcp = h1; qam += h2; }                   // +y+z / -y-z
                else { qap += h1; qcm = h2; }                                // +y-z / -y+z
                // corners: only c_z = 0 directions reach a diagonal tile, so the target plane is this plane
                if ((p == 3 || p == 4) && store_h && (lane_lo || lane_hi) && (row_lo || row_hi)) {
                    const bool main_diag = lane_hi == row_hi;
                    if ((p == 3) == main_diag) {
                        const int kk = opaque(k);
                        const unsigned e_xy = unsigned(kk * ro.s_xy) + ((row_hi ? btyp : btym) * ntx + (lane_hi ? btxp : btxm)) * 4 + (row_hi ? (lane_hi ? 0 : 1) : (lane_hi ? 2 : 3));
                        ro.xy[e_xy + zl * psxy] = lane_hi ? h1 : h2;
                    }
                }
            });
        const T p0 = qa0, pp = qap, pm = qam;               // complete for plane z-1
        qa0 = qb0; qb0 = qc0;
        qap = qbp; qbp = qcp;
        qam = qbm; qbm = qcm;
        SUup[0] = pp;
        SUum[0] = pm;
        __syncwarp();
        if (lane_lo) mbar_arrive(rowpub + sg * 2 * TY + k * TY + ty);

        // ---- the y-edge exports need nothing from the other warps ----
        if ((row_lo || row_hi) && store_rho) {
            const int kk = opaque(k);
            const bool lo = opaque(ty) == 0;
            const unsigned e_y = unsigned(kk * ro.s_y) + ((lo ? btym : btyp) * 2 + (lo ? 1 : 0)) * nx + x0 + tx;
            ro.y[e_y + zt * psy] = lo ? pm : pp;
        }
        {   // the rows above and below (same component) have published this plane
            unsigned long long* nb = rowpub + sg * 2 * TY + k * TY + ty;
            if (row_lo) mbar_wait(nb + 1, ph);
            else if (row_hi) mbar_wait(nb - 1, ph);
            else mbar_wait2(nb - 1, nb + 1, ph);
        }

        // ---- y stage of the gather: the tile's own edge rows / columns, and the exports across its x edges ----
        {
            T out = p0;
            if (!row_lo) out += SUup[-RW];
            if (!row_hi) out += SUum[RW];
            if ((row_lo || row_hi) && store_rho) {
                const int kk = opaque(k);
                const unsigned e_r = unsigned(kk * ro.s_y) + (bty * 2 + (opaque(ty) == 0 ? 0 : 1)) * nx + x0 + tx;
                ro.er[e_r + zt * psy] = out;
            }
            if (lane_lo || lane_hi) {
                const int vc = lane_lo ? -1 : 1;
                T a_0 = exs[1];
                if (!row_lo) a_0 += SUup[vc - RW];
                if (!row_hi) a_0 += SUum[vc + RW];
                const T hout = exs[3] + exs[0];
                exs[3] = exs[4] + a_0;
                exs[4] = exs[2];
                if (store_rho) {
                    const int kk = opaque(k);
                    const unsigned e_c = unsigned(kk * ro.s_x) + ((bty * ntx + btx) * 2 + (lane_lo ? 0 : 1)) * TY + ty;
                    ro.ec[e_c + zt * psx] = out;
                    const unsigned e_x = unsigned(kk * ro.s_x) + ((bty * ntx + (lane_lo ? btxm : btxp)) * 2 + (lane_lo ? 1 : 0)) * TY + ty;
                    ro.x[e_x + zt * psx] = hout;
                }
            }
        }
        zt = zl;
        zl = zl + 1 == nz ? 0 : zl + 1;
    }

    if (DIAG) {
        // per-CTA partial sums {mass_r, mass_b, P_x, P_y, P_z}: warp shuffles, then the 2 TY warp partials in a fixed order
        double v[4] = {dacc[0], dacc[NC], dacc[2 * NC], dacc[3 * NC]};
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], off);
        asm volatile("bar.sync 9, %0;" ::"n"(NC) : "memory");              // every consumer has read its accumulators
        double* wp = reinterpret_cast<double*>(smem_halo + L::DIAG_BYTE_OFF);
        if (tx == 0) { const int w = t / 32; wp[w * 4 + 0] = v[0]; wp[w * 4 + 1] = v[1]; wp[w * 4 + 2] = v[2]; wp[w * 4 + 3] = v[3]; }
        asm volatile("bar.sync 9, %0;" ::"n"(NC) : "memory");
        if (t < 5) {
            double s = 0.0;
            if (t < 2) { for (int w = 0; w < TY; ++w) s += wp[(t * TY + w) * 4]; }
            else { for (int w = 0; w < 2 * TY; ++w) s += wp[w * 4 + t - 1]; }
            const long long cta = blockIdx.x + (long long)gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z);
            diag_part[cta * 5 + t] = s;
        }
    }
}

// x-halo arrays of a population buffer (header): one thread per (plane q' = 2 j + k, z, tile_x, y')
template <typename T>
__global__ void __launch_bounds__(256) k_fill_xhalo(const T* __restrict__ h, T* __restrict__ hx, long long NP, int nx, int ny, int nz) {
    const int ntx = nx / 32;
    const long long total = (long long)2 * NHALO * nz * ntx * ny;
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= total) return;
    const int yp = int(e % ny);
    const int b = int((e / ny) % ntx);
    const int z = int((e / ((long long)ny * ntx)) % nz);
    const int qp = int(e / ((long long)ny * ntx * nz));
    const int j = qp / 2, k = qp % 2;
    const int i = j < 2 ? j + 1 : j + 5;
    const int cx = dir_cx(i), cy = dir_cy(i);
    int y = yp - cy;
    y = y < 0 ? y + ny : (y >= ny ? y - ny : y);
    const int x = b * 32 + (cx > 0 ? 31 : 0);
    hx[e] = h[(long long)pop_plane(k, i) * NP + ((long long)z * ny + y) * nx + x];
}

// frame-density arrays from a full density field rho[k][NP] (the initial state): er / ec = the edge rows / columns, x / y / xy = 0
template <typename T>
__global__ void __launch_bounds__(256) k_edges_from_rho(const T* __restrict__ rho, long long NP, EdgeView<T> ev, int nx, int ny, int nz, int TYv) {
    const long long N = (long long)nx * ny * nz;
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    const int x = int(n % nx), y = int((n / nx) % ny), z = int(n / ((long long)nx * ny));
    const int ntx = nx / 32, nty = ny / TYv;
    const int btx = x / 32, lx = x % 32, bty = y / TYv, ly = y % TYv;
    const long long psx = (long long)nty * ntx * 2 * TYv, psy = (long long)nty * 2 * nx;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const T v = rho[k * NP + n];
        if (ly == 0 || ly == TYv - 1) ev.er[k * ev.s_y + z * psy + (bty * 2 + (ly != 0)) * nx + x] = v;
        if (lx == 0 || lx == 31) ev.ec[k * ev.s_x + z * psx + ((bty * ntx + btx) * 2 + (lx != 0)) * TYv + ly] = v;
    }
}

}  // namespace lb
