// lb_tma.cuh -- the fused one-pass time step with TMA-staged populations (the hot kernel on B200).
//
// Same algorithm and same state convention as lb_onepass.cuh (h-state, pull streaming, density carried
// from step to step through the four single-writer arrays rho_in / rho_x / rho_y / rho_xy), but the
// 38 population planes of a tile are brought into shared memory by the TMA unit instead of by 38
// per-thread loads, and one thread handles one (node, component) instead of one node:
//   * one producer warp per CTA issues, per z plane, 38 `cp.async.bulk.tensor.4d` box loads (one per
//     population plane, box = tile shifted by -c_i in y and z) that complete on an mbarrier; the
//     consumer threads then read their 19 values with LDS at fixed offsets: no per-thread address
//     arithmetic, no registers in flight, and the prefetch distance is a whole plane whatever the
//     occupancy is;
//   * measured on B200: a TMA box whose innermost start is not 16-byte aligned
//     raises an illegal-instruction fault, so the x shift cannot be given to the TMA.  Directions with
//     c_x != 0 are loaded as an ALIGNED box that is PADX = 16/sizeof(T) elements wider, and the consumer
//     applies the shift in its LDS address (free);
//   * the TMA zero-fills out-of-range box parts and does not wrap.  x: tiles at the box
//     boundary load, per direction with c_x != 0, one more box (PADX x TY) holding the wrapped column,
//     and the lane next to the edge reads that box instead (a different base offset, same instruction).
//     y: the one warp whose row lies beyond the edge re-loads its 5 affected populations with plain loads.
//     z wraps in the box coordinate;
//   * consumers copy the stage into registers and release it at once, so one stage buffers a whole
//     plane of prefetch; post-collision values are stored straight from registers (aligned, coalesced);
//   * the two threads of a node exchange rho^k, j^k through shared memory (common velocity, S4) with a
//     64-thread named barrier per tile row; the y stage of the density gather is double-buffered behind
//     one split-phase mbarrier per plane (arrive, independent stores, wait); the stage hand-off is
//     mbarriers only;
//   * three more warps of the producer group assemble the density ring two planes ahead of its use from tabulated
//     piece lists (cp.async into landing slots, then the fixed-order sums);
//   * the producer warp group hands registers to the consumers (setmaxnreg): 16 consumer warps at 104
//     registers, producer group at 64.
#pragma once
#include <cuda.h>

#include "lb_lattice.cuh"
#include "lb_onepass.cuh"

namespace lb {

// ---- PTX wrappers ----------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return static_cast<unsigned>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(void* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, 0x989680;\n\t"
        "@P1 bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// box load: coordinates (x, y, z, plane); x * sizeof(T) must be a multiple of 16 (see header)
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, void* bar, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
// the same box, into L2 only
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* tm, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
// plain global stores through a pointer the compiler must treat as opaque (see the running store pointer in the kernel)
__device__ __forceinline__ void st_global(double* p, double v) { asm volatile("st.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }
__device__ __forceinline__ void st_global(float* p, float v) { asm volatile("st.global.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }
// products and sums the compiler may not contract into an fma
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
template <int ID, int COUNT>
__device__ __forceinline__ void named_barrier() { asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(COUNT) : "memory"); }

// ---- shared-memory layout -----------------------------------------------------------------------------
template <typename T, int TY>
struct TmaLayout {
    static constexpr int TX = 32, NT = TX * TY;
    static constexpr int PADX = 16 / int(sizeof(T));                   // elements per 16 bytes
    static constexpr int W = TX + PADX;                                // row length of a wide (c_x != 0) slot
    static constexpr int RW = TX + 2, RH = TY + 2, RS = RW * RH;       // density ring plane: tile + one-node frame
    static constexpr int SUP = TY * RW;                                // one y-stage plane: tile rows with an x frame
    __host__ __device__ static constexpr int align128(int elems) { return (elems * int(sizeof(T)) + 127) / 128 * 128 / int(sizeof(T)); }
    static constexpr int XC = align128(W * TY);                        // offset of the wrapped-column box inside a wide slot (128-byte aligned)
    static constexpr int NA = align128(NT), WA = align128(XC + PADX * TY);    // slot sizes: narrow (c_x = 0) and wide (+ wrapped column), 128-byte multiples
    // number of wide slots before direction i (the directions with c_x != 0 are 1, 2, 7..14)
    __host__ __device__ static constexpr int wide_before(int i) { return (i > 1) + (i > 2) + (i > 7 ? (i - 7 < 8 ? i - 7 : 8) : 0); }
    __host__ __device__ static constexpr int slot_off(int q) {         // element offset of population plane q = k*19 + i
        return (q / Q) * (9 * NA + 10 * WA) + (q % Q - wide_before(q % Q)) * NA + wide_before(q % Q) * WA;
    }
    static constexpr int STAGE = 0;
    static constexpr int STAGE_ELEMS = slot_off(NPOP);
    static constexpr unsigned STAGE_TX_BYTES = unsigned(2 * (9 * NT + 10 * W * TY) * sizeof(T));   // bytes the 38 boxes deliver
    static constexpr unsigned XCOL_TX_BYTES = unsigned(2 * 5 * PADX * TY * sizeof(T));             // ... plus the 10 wrapped-column boxes of one x side
    static constexpr int RING = STAGE + STAGE_ELEMS;                   // [4][2][RS]      rho(t), planes z-1..z+2
    static constexpr int SU = RING + 8 * RS;                           // [2][2][2][SUP]  double-buffered z-summed Up, Um per component
    static constexpr int XM = SU + 8 * SUP;                           // [2][NT][4]      rho^k, j^k of every node, exchanged between the two components' threads
    // ring pieces: every ring position has an `in` piece; the positions in the 4 columns / 4 rows next to a tile edge
    // also have an x / y piece, the 16 where they cross an xy piece
    static constexpr int NEX = 4 * RH, NEY = 4 * RW, NEXY = 16;
    static constexpr int RP_IN = XM + 8 * NT;                          // [2][RS]    landing slots of the pieces (cp.async), per component
    static constexpr int RP_X = RP_IN + 2 * RS;                        // [2][NEX]
    static constexpr int RP_Y = RP_X + 2 * NEX;                        // [2][NEY]
    static constexpr int RP_XY = RP_Y + 2 * NEY;                       // [2][NEXY]
    static constexpr int END = RP_XY + 2 * NEXY;
    static constexpr size_t TAB_BYTE_OFF = (size_t(END) * sizeof(T) + 15) / 16 * 16;
    // int tables: T_IN[RS] offset of the in piece inside a plane; T_PK[RS] packed list indices (x | y << 8 | xy << 16, 255 = none);
    // T_X[NEX], T_Y[NEY], T_XY[NEXY] offsets of the edge pieces inside their arrays' planes
    static constexpr int T_IN = 0, T_PK = RS, T_X = 2 * RS, T_Y = T_X + NEX, T_XY = T_Y + NEY, T_END = T_XY + NEXY;
    static constexpr size_t BAR_BYTE_OFF = (TAB_BYTE_OFF + size_t(T_END) * sizeof(int) + 15) / 16 * 16;
    static constexpr size_t BYTES = BAR_BYTE_OFF + 8 * sizeof(unsigned long long);
};


#ifdef LB_TMA_TRACE
__device__ long long g_trace[64 * 16];
#define TRACE(cond, it, slot) do { if ((cond) && blockIdx.x == 1 && blockIdx.y == 1 && blockIdx.z == 0 && (it) >= 0 && (it) < 64) g_trace[(it) * 16 + (slot)] = clock64(); } while (0)
#else
#define TRACE(cond, it, slot) do { } while (0)
#endif

// ---- the kernel ------------------------------------------------------------------------------------------
// Threads: 2*NT consumers (component k = t / NT, node (tx, ty) = ((t % NT) % 32, (t % NT) / 32): one warp per
// tile row and component) followed by one producer warp group (only its first warp works).  The producer
// group gives its registers to the consumers (setmaxnreg), which is why it is a whole warp group.
template <typename T, bool HAS_SOLID, int TY>
__global__ void __launch_bounds__(2 * 32 * TY + 128, TY <= 4 ? 2 : 1)
k_step_tma(const __grid_constant__ CUtensorMap tm_n, const __grid_constant__ CUtensorMap tm_w,
           const __grid_constant__ CUtensorMap tm_c, const T* __restrict__ h, T* __restrict__ g, const unsigned* __restrict__ links,
           const RhoView<T> ri, const RhoView<T> ro, long long NP, int nx, int ny, int nz, int zc,
           T om_r, T om_b, T G) {
    using L = TmaLayout<T, TY>;
    constexpr int TX = L::TX, NT = L::NT, NC = 2 * NT, RW = L::RW, RS = L::RS, SUP = L::SUP, W = L::W, PADX = L::PADX;
    static_assert(RS <= 2 * NT, "ring fill: at most two positions per consumer thread");
    static_assert(2 * L::NEX <= 96 && 2 * L::NEXY <= 96, "one ring thread per x / xy piece");
    static_assert(TY >= 2 && TY <= 8, "one named barrier per tile row (ids 1..TY)");
    // register hand-over between the warp groups: (2*NT + 128) threads start with 65536 / threads registers each
    constexpr int CTAS_PER_SM = TY <= 4 ? 2 : 1;
    constexpr int START_REGS = (65536 / ((NC + 128) * CTAS_PER_SM)) / 8 * 8;
    constexpr int PRODUCER_REGS = TY <= 4 ? 32 : 64;
    constexpr int CONSUMER_REGS = (START_REGS + (START_REGS - PRODUCER_REGS) * 128 / NC) / 8 * 8;
    extern __shared__ __align__(1024) unsigned char smem_tma[];
    T* sm = reinterpret_cast<T*>(smem_tma);
    T* stage = sm + L::STAGE;
    T* ring = sm + L::RING;
    T* SUb = sm + L::SU;
    T* xm = sm + L::XM;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_tma + L::BAR_BYTE_OFF);
    unsigned long long* full = bars;          // the 38 boxes of the next plane have landed (tx bytes)
    unsigned long long* done = bars + 2;      // every consumer warp has copied its part of the stage into registers
    unsigned long long* pub = bars + 3;       // every consumer warp has published its y-stage inputs of this plane
    unsigned long long* rdy = bars + 4;       // the producer warp has assembled the density ring plane this iteration needs
    int* tab = reinterpret_cast<int*>(smem_tma + L::TAB_BYTE_OFF);

    const int t = threadIdx.x;
    const int ntx = nx / TX, nty = ny / TY;
    const int btx = blockIdx.x, bty = blockIdx.y;
    const int x0 = btx * TX, y0 = bty * TY;
    const int z0 = blockIdx.z * zc;
    const int z1 = min(z0 + zc, nz);
    const int niter = z1 - z0 + 2;            // planes z0-1 .. z1; the first and the last are re-collided only
    const long long pl = (long long)nx * ny;
    const bool wrap_xlo = btx == 0, wrap_xhi = btx == ntx - 1;             // the TMA zero-fills outside the box: x wraps with an
                                                                           // extra box per direction, y with consumer loads
    auto wrapz = [&](int p) { p %= nz; return p < 0 ? p + nz : p; };

    if (t == 0) {
        mbar_init(full, 1);
        mbar_init(done, 2 * TY);
        mbar_init(pub, 2 * TY);
        mbar_init(rdy, 3);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // ---- density ring bookkeeping: ring position pos (tile + one-node frame) of either component is the sum
    //      ((in + x) + y) + xy of up to four single-writer pieces (lb_onepass.cuh); where they live, tabulated once ----
    for (int pos = t; pos < RS; pos += blockDim.x) {
        const int rx = pos % RW - 1, ry = pos / RW - 1;
        const int txm = btx == 0 ? ntx - 1 : btx - 1, txp = btx == ntx - 1 ? 0 : btx + 1;
        const int tym = bty == 0 ? nty - 1 : bty - 1, typ = bty == nty - 1 ? 0 : bty + 1;
        const int otx = rx < 0 ? txm : (rx >= TX ? txp : btx), oty = ry < 0 ? tym : (ry >= TY ? typ : bty);
        const int lx = rx < 0 ? TX - 1 : (rx >= TX ? 0 : rx), ly = ry < 0 ? TY - 1 : (ry >= TY ? 0 : ry);
        const int c4 = rx == -1 ? 0 : (rx == 0 ? 1 : (rx == TX - 1 ? 2 : (rx == TX ? 3 : -1)));   // edge column / row of the tile grid
        const int r4 = ry == -1 ? 0 : (ry == 0 ? 1 : (ry == TY - 1 ? 2 : (ry == TY ? 3 : -1)));
        tab[L::T_IN + pos] = (oty * TY + ly) * nx + otx * TX + lx;
        int pk = 0xFFFFFF;
        if (c4 >= 0) {
            const int m = c4 * L::RH + ry + 1;
            tab[L::T_X + m] = ((oty * ntx + otx) * 2 + (lx != 0)) * TY + ly;
            pk = (pk & ~0xFF) | m;
        }
        if (r4 >= 0) {
            const int m = r4 * RW + rx + 1;
            tab[L::T_Y + m] = (oty * 2 + (ly != 0)) * nx + otx * TX + lx;
            pk = (pk & ~0xFF00) | (m << 8);
        }
        if (c4 >= 0 && r4 >= 0) {
            const int m = r4 * 4 + c4;
            tab[L::T_XY + m] = (oty * ntx + otx) * 4 + (ly != 0) * 2 + (lx != 0);
            pk = (pk & ~0xFF0000) | (m << 16);
        }
        tab[L::T_PK + pos] = pk;
    }
    __syncthreads();

    // =================================== producer warp ===================================
    if (t >= NC) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
        if (t >= NC + 32) {
            // ---- ring warps (3): assemble the density ring, one plane per iteration, two planes ahead of its use ----
            const int r = t - NC - 32;
            constexpr int NR = 96;
            const long long psx_ = (long long)nty * ntx * 2 * TY, psy_ = (long long)nty * 2 * nx, psxy_ = (long long)nty * ntx * 4;
            T* s_in = sm + L::RP_IN;
            T* s_x = sm + L::RP_X;
            T* s_y = sm + L::RP_Y;
            T* s_xy = sm + L::RP_XY;
            auto ring_sync = [&]() { asm volatile("bar.sync %0, %1;" ::"n"(TY + 2), "n"(NR) : "memory"); };
            // ask for the pieces of ring plane rp (= box plane z0 - 2 + rp): asynchronous, no registers in flight
            auto ring_fetch = [&](int rp) {
                const long long zp = wrapz(z0 - 2 + rp);
#pragma unroll
                for (int kk = 0; kk < 2; ++kk) {
                    const T* b_in = ri.in + kk * ri.s_in + zp * pl;
                    for (int pos = r; pos < RS; pos += NR) cp_async<sizeof(T)>(s_in + kk * RS + pos, b_in + tab[L::T_IN + pos]);
                    const T* b_y = ri.y + kk * ri.s_y + zp * psy_;
                    for (int m = r; m < L::NEY; m += NR) cp_async<sizeof(T)>(s_y + kk * L::NEY + m, b_y + tab[L::T_Y + m]);
                }
                if (r < 2 * L::NEX) {
                    const int kk = r >= L::NEX, m = r - kk * L::NEX;
                    cp_async<sizeof(T)>(s_x + r, ri.x + kk * ri.s_x + zp * psx_ + tab[L::T_X + m]);
                }
                if (r >= NR - 2 * L::NEXY) {
                    const int q = r - (NR - 2 * L::NEXY), kk = q >= L::NEXY, m = q - kk * L::NEXY;
                    cp_async<sizeof(T)>(s_xy + q, ri.xy + kk * ri.s_xy + zp * psxy_ + tab[L::T_XY + m]);
                }
                cp_async_commit();
            };
            // ... and add them up in the fixed order ((in + x) + y) + xy once they have landed
            auto ring_assemble = [&](int rp) {
                cp_async_wait<0>();
                TRACE(r == 0, rp - 2, 14);
                ring_sync();                                               // every ring thread's pieces are in
                TRACE(r == 0, rp - 2, 15);
                T* dst = ring + (rp & 3) * 2 * RS;
#pragma unroll
                for (int kk = 0; kk < 2; ++kk)
                    for (int pos = r; pos < RS; pos += NR) {
                        T v = s_in[kk * RS + pos];
                        const int pk = tab[L::T_PK + pos];
                        if (pk != 0xFFFFFF) {
                            const int ix = pk & 255, iy = (pk >> 8) & 255, ixy = (pk >> 16) & 255;
                            if (ix != 255) v += s_x[kk * L::NEX + ix];
                            if (iy != 255) v += s_y[kk * L::NEY + iy];
                            if (ixy != 255) v += s_xy[kk * L::NEXY + ixy];
                        }
                        dst[kk * RS + pos] = v;
                    }
                TRACE(r == 0, rp - 2, 11);
                ring_sync();                                               // the landing slots may be overwritten
            };
            for (int rp = 0; rp < 2; ++rp) {                                // iteration 0 needs ring planes 0, 1, 2
                ring_fetch(rp);
                ring_assemble(rp);
            }
            ring_fetch(2);
            for (int j = 0; j < niter; ++j) {
                // ring plane j+2 (the z+1 neighbour plane of iteration j): its slot held plane j-2, last read in iteration
                // j-2, which every consumer warp had left when it arrived on done(j-1)
                if (j > 0) mbar_wait(done, (j - 1) & 1);
                TRACE(r == 0, j, 8);
                ring_assemble(j + 2);
                __syncwarp();
                if ((r & 31) == 0) mbar_arrive(rdy);
                TRACE(r == 0, j, 9);
                if (j + 3 <= niter + 1) ring_fetch(j + 3);
                TRACE(r == 0, j, 10);
            }
            return;
        }
        // ---- TMA warp ----
        const int lane = t - NC;
        for (int j = 0; j < niter; ++j) {
            const int z = z0 - 1 + j;
            const int zw[3] = {wrapz(z - 1), wrapz(z), wrapz(z + 1)};
            if (lane == 0) {
                if (j > 0) mbar_wait(done, (j - 1) & 1);
                TRACE(true, j, 12);
                mbar_expect_tx(full, L::STAGE_TX_BYTES + (wrap_xlo ? L::XCOL_TX_BYTES : 0u) + (wrap_xhi ? L::XCOL_TX_BYTES : 0u));
#pragma unroll
                for (int q = 0; q < NPOP; ++q) {
                    const int i = q % Q;
                    const int zq = zw[1 - dir_cz(i)];                       // f_i(x) = h_i(x - c_i)
                    T* slot = stage + L::slot_off(q);
                    if (dir_cx(i) == 0) tma_load_4d(slot, &tm_n, full, x0, y0 - dir_cy(i), zq, q);
                    else {
                        tma_load_4d(slot, &tm_w, full, dir_cx(i) > 0 ? x0 - PADX : x0, y0 - dir_cy(i), zq, q);
                        // the column beyond the box edge: columns nx-PADX..nx-1 for c_x > 0, 0..PADX-1 for c_x < 0
                        if (dir_cx(i) > 0 && wrap_xlo) tma_load_4d(slot + L::XC, &tm_c, full, nx - PADX, y0 - dir_cy(i), zq, q);
                        if (dir_cx(i) < 0 && wrap_xhi) tma_load_4d(slot + L::XC, &tm_c, full, 0, y0 - dir_cy(i), zq, q);
                    }
                }
                if (j + 1 < niter) {                                        // the plane after that: DRAM -> L2 now, so that its
                    const int zn[3] = {zw[1], zw[2], wrapz(z + 2)};         // box loads (one stage, issued late) hit in L2
#pragma unroll
                    for (int q = 0; q < NPOP; ++q) {
                        const int i = q % Q;
                        if (dir_cx(i) == 0) tma_prefetch_4d(&tm_n, x0, y0 - dir_cy(i), zn[1 - dir_cz(i)], q);
                        else tma_prefetch_4d(&tm_w, dir_cx(i) > 0 ? x0 - PADX : x0, y0 - dir_cy(i), zn[1 - dir_cz(i)], q);
                    }
                }
            }
            TRACE(lane == 0, j, 13);
            __syncwarp();
        }
        return;
    }

    // =================================== consumers ===================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
    const int k = t / NT;                                                  // component of this thread (warp-uniform)
    const int tl = t - k * NT;
    const int tx = tl % TX, ty = tl / TX;
    const int x = x0 + tx, y = y0 + ty;
    const int own_xy = y * nx + x;
    const int own_r = (ty + 1) * RW + tx + 1;                              // ring position (tile + frame)
    const int own_s = ty * RW + tx + 1;                                    // y-stage plane position (x frame only)
    const long long psx = (long long)nty * ntx * 2 * TY, psy = (long long)nty * 2 * nx, psxy = (long long)nty * ntx * 4;
    const int btxm = btx == 0 ? ntx - 1 : btx - 1, btxp = btx == ntx - 1 ? 0 : btx + 1;
    const int btym = bty == 0 ? nty - 1 : bty - 1, btyp = bty == nty - 1 ? 0 : bty + 1;
    const T zero = T(0);
    const T om_own = k == 0 ? om_r : om_b, om_oth = k == 0 ? om_b : om_r;
    const T omc = T(1) - om_own;
    const T* stage_k = stage + k * (9 * L::NA + 10 * L::WA);
    const T* hk = h + (long long)k * Q * NP;
    T* gk = g + (long long)k * Q * NP + own_xy;
    const T* ring_o = ring + (1 - k) * RS;                                 // the OTHER component's density (S2)
    T* SUk = SUb + k * 2 * SUP;
    T* ro_in = ro.in + k * ro.s_in + own_xy;
    const bool lane_lo = tx == 0, lane_hi = tx == TX - 1, row_lo = ty == 0, row_hi = ty == TY - 1;
    // where this thread finds f_i = h_i(x - c_i) inside slot i, by c_x: the x shift is applied here; the lane next to the
    // box edge reads the wrapped-column box instead
    const int rd0 = ty * TX + tx;
    const int rdp = (wrap_xlo && lane_lo) ? L::XC + ty * PADX + PADX - 1 : ty * W + tx + PADX - 1;
    const int rdm = (wrap_xhi && lane_hi) ? L::XC + ty * PADX : ty * W + tx + 1;
    const bool wrap_ylo = bty == 0 && row_lo, wrap_yhi = bty == nty - 1 && row_hi;   // warp-uniform

    // ---- per-thread state carried along z ----
    // z pipelines of the density gather, one per y class of the row sums (U0: c_y = 0, Up: c_y = +1, Um: c_y = -1):
    // [0] = V_+1(z-2) + V_0(z-1), [1] = V_+1(z-1); adding V_-1(z) completes plane z-1
    T acc0[2] = {zero, zero}, accp[2] = {zero, zero}, accm[2] = {zero, zero};
    T col_acc[2] = {zero, zero};     // the same for the export across the tile's x edge (lanes tx = 0 and TX-1)

    int zl = wrapz(z0 - 1), zt = wrapz(z0 - 2);         // this plane / the plane the gathered density belongs to
    unsigned lk = 0;
    if (HAS_SOLID) lk = __ldg(links + (long long)zl * pl + own_xy);

#pragma unroll 1
    for (int it = 0; it < niter; ++it) {
        const long long zoff = (long long)zl * pl;
        const bool store_h = it >= 1 && it <= niter - 2;
        const bool store_rho = it >= 2;                 // target plane z-1 lies in [z0, z1)
        const int s0 = (it + 1) & 3;                    // ring slot of plane z
        const bool fluid = !HAS_SOLID || !(lk & OP_SOLID_BIT);   // nothing happens inside a particle
        T* SU = SUk + (it & 1) * 4 * SUP;

        // ---- pull: the stage holds h_i(x - c_i) for the whole tile (Eq. 5, periodic) ----
        TRACE(t == 0, it, 0);
        mbar_wait(full, it & 1);
        TRACE(t == 0, it, 1);
        mbar_wait(rdy, it & 1);                         // density ring planes z-1, z, z+1 are in place (before `done`: the producer
                                                        // must not get two phases ahead of any waiter)
        TRACE(t == 0, it, 2);
        T f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = stage_k[L::slot_off(i) + (dir_cx(i) == 0 ? rd0 : (dir_cx(i) > 0 ? rdp : rdm))];
        if (wrap_ylo || wrap_yhi) {                     // the row beyond the box edge in y (one warp of a boundary tile): plain loads
            const int gy = wrap_ylo ? ny - 1 : 0;
            const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
            const long long zs[3] = {(long long)zt * pl, zoff, (long long)(zl + 1 == nz ? 0 : zl + 1) * pl};
#pragma unroll
            for (int i = 1; i < Q; ++i)
                if (dir_cy(i) != 0) {
                    const T v = __ldg(hk + (long long)i * NP + zs[1 - dir_cz(i)] + (long long)gy * nx + xs[1 - dir_cx(i)]);
                    if ((dir_cy(i) > 0 && wrap_ylo) || (dir_cy(i) < 0 && wrap_yhi)) f[i] = v;
                }
        }
        if (HAS_SOLID && (lk & 0x7FFFEu)) {             // halfway bounce-back (Eq. 23-24, u_b = 0): f_i(x) = h_opp(i)(x) when x - c_i is solid
#pragma unroll
            for (int i = 1; i < Q; ++i)
                if (lk >> dir_opp(i) & 1u) f[i] = __ldg(hk + (long long)dir_opp(i) * NP + zoff + own_xy);
        }
        __syncwarp();
        TRACE(t == 0, it, 3);
        if (lane_lo) mbar_arrive(done);                 // the producer may refill the stage with the next plane

        // ---- moments of this component (Eq. 6-7), exchanged with the other component's thread of the same node ----
        T rho = zero, jx = zero, jy = zero, jz = zero;
        if (fluid) moments19<T>(f, rho, jx, jy, jz);
        else {
#pragma unroll
            for (int i = 0; i < Q; ++i) f[i] = zero;
        }
        {
            T* mine = xm + (k * NT + tl) * 4;
            mine[0] = rho; mine[1] = jx; mine[2] = jy; mine[3] = jz;
        }
        asm volatile("bar.sync %0, 64;" ::"r"(ty + 1) : "memory");         // the two warps (red, blue) of this tile row
        T ux = zero, uy = zero, uz = zero, ex = zero, ey = zero, ez = zero;
        if (fluid) {
            const T* other = xm + ((1 - k) * NT + tl) * 4;
            const T orho = other[0], ojx = other[1], ojy = other[2], ojz = other[3];
            // common velocity (S4): u' = (om_r j^r + om_b j^b) / (om_r rho^r + om_b rho^b).  Both threads of the node must
            // get the same bits: separately rounded products and one sum are commutative, a contracted fma is not.
            const T den = add_rn(mul_rn(om_own, rho), mul_rn(om_oth, orho));
            const T inv = den != zero ? T(1) / den : zero;
            ux = add_rn(mul_rn(om_own, jx), mul_rn(om_oth, ojx)) * inv;
            uy = add_rn(mul_rn(om_own, jy), mul_rn(om_oth, ojy)) * inv;
            uz = add_rn(mul_rn(om_own, jz), mul_rn(om_oth, ojz)) * inv;
            // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6); a solid neighbour counts psi = 0 (S7)
            T d[9];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                T vp = ring_o[sp * 2 * RS + own_r + pair_cy(p) * RW + pair_cx(p)];
                T vm = ring_o[sm_ * 2 * RS + own_r - pair_cy(p) * RW - pair_cx(p)];
                if (HAS_SOLID) {
                    if (lk >> (2 * p + 1) & 1u) vp = zero;
                    if (lk >> (2 * p + 2) & 1u) vm = zero;
                }
                d[p] = w_pair<T>(p) * (vp - vm);
            }
            const T gx = (((d[0] + d[3]) + d[4]) + d[5]) + d[6];
            const T gy = (((d[1] + d[3]) - d[4]) + d[7]) + d[8];
            const T gz = (((d[2] + d[5]) - d[6]) + d[7]) - d[8];
            ex = ux - G * gx; ey = uy - G * gy; ez = uz - G * gz;
        }

        // ---- BGK collision with exact-difference forcing (Eq. 1, Eq. 10, S5), and, pair by pair as the post-collision values
        //      appear: their (aligned, coalesced) stores and the x stage of the density gather
        //      rho(y, t+1) = sum_i h_i(y - c_i): x by warp shuffles, z by register pipelines, y through shared memory.
        //      A solid node runs the same instructions on zeros (the shuffles need every lane) and stores nothing. ----
        T u0[3] = {zero, zero, zero};                    // row sums by c_z, c_y = 0
        T ee[3] = {zero, zero, zero};                    // on lanes tx = 0 / TX-1: what leaves the tile in x with c_y = 0
        T up[3] = {zero, zero, zero}, um[3] = {zero, zero, zero};   // c_y = +1 / -1
        T* SUup = SU;                                    // interior: Up summed over z (plane z-1); x frame: Up[c_z = 0] of the virtual column, plane z
        T* SUum = SU + SUP;
        T bs = zero;                                     // bounced-back arrivals of the next step come from this node
        const bool do_store = fluid && store_h;
        T* o = gk + zoff;                                // values arrive in direction order: a running pointer
        auto put = [&](T v) {
            if (do_store) st_global(o, v);
            o += NP;
            asm volatile("" : "+l"(o));                  // keep it a pointer: ptxas otherwise re-derives every address from scratch
        };
        collide19_pairs<T>(f, rho, omc, ux, uy, uz, ex, ey, ez,
            [&](T h0) { put(h0); u0[1] = h0; },
            [&](int p, T h1, T h2) {
                put(h1);
                put(h2);
                if (HAS_SOLID) {
                    if (lk >> (2 * p + 1) & 1u) bs += h1;
                    if (lk >> (2 * p + 2) & 1u) bs += h2;
                }
                T l = zero, r = zero;
                if (p == 0 || (p >= 3 && p <= 6)) { l = __shfl_up_sync(0xffffffffu, h1, 1); r = __shfl_down_sync(0xffffffffu, h2, 1); }
                if (p == 0) {                                              // +x / -x
                    if (!lane_lo) u0[1] += l;
                    if (!lane_hi) u0[1] += r;
                    ee[1] = lane_hi ? h1 : h2;
                } else if (p == 1) { up[1] = h1; um[1] = h2; }              // +y / -y
                else if (p == 2) { u0[2] = h1; u0[0] = h2; }                // +z / -z
                else if (p == 3) {                                         // +x+y / -x-y
                    up[1] += lane_lo ? zero : l;
                    um[1] += lane_hi ? zero : r;
                    if (lane_hi) SUup[own_s + 1] = h1;
                    if (lane_lo) SUum[own_s - 1] = h2;
                } else if (p == 4) {                                       // +x-y / -x+y
                    um[1] += lane_lo ? zero : l;
                    up[1] += lane_hi ? zero : r;
                    if (lane_hi) SUum[own_s + 1] = h1;
                    if (lane_lo) SUup[own_s - 1] = h2;
                } else if (p == 5) {                                       // +x+z / -x-z
                    if (!lane_lo) u0[2] += l;
                    if (!lane_hi) u0[0] += r;
                    if (lane_hi) ee[2] = h1;
                    if (lane_lo) ee[0] = h2;
                } else if (p == 6) {                                       // +x-z / -x+z
                    if (!lane_lo) u0[0] += l;
                    if (!lane_hi) u0[2] += r;
                    if (lane_hi) ee[0] = h1;
                    if (lane_lo) ee[2] = h2;
                } else if (p == 7) { up[2] = h1; um[0] = h2; }              // +y+z / -y-z
                else { up[0] = h1; um[2] = h2; }                           // +y-z / -y+z
                // corners: only c_z = 0 directions reach a diagonal tile, so the target plane is this plane
                if ((p == 3 || p == 4) && store_h && (lane_lo || lane_hi) && (row_lo || row_hi)) {
                    T* cxy = ro.xy + k * ro.s_xy + zl * psxy;
                    if (p == 3 && lane_hi && row_hi) cxy[(btyp * ntx + btxp) * 4 + 0] = h1;     // +x+y
                    if (p == 3 && lane_lo && row_lo) cxy[(btym * ntx + btxm) * 4 + 3] = h2;     // -x-y
                    if (p == 4 && lane_hi && row_lo) cxy[(btym * ntx + btxp) * 4 + 2] = h1;     // +x-y
                    if (p == 4 && lane_lo && row_hi) cxy[(btyp * ntx + btxm) * 4 + 1] = h2;     // -x+y
                }
            });
        if (HAS_SOLID) u0[1] += bs;
        const T p0 = acc0[0] + u0[0], pp = accp[0] + up[0], pm = accm[0] + um[0];   // complete for plane z-1
        acc0[0] = acc0[1] + u0[1]; acc0[1] = u0[2];
        accp[0] = accp[1] + up[1]; accp[1] = up[2];
        accm[0] = accm[1] + um[1]; accm[1] = um[2];
        SUup[own_s] = pp;
        SUum[own_s] = pm;
        __syncwarp();
        if (lane_lo) mbar_arrive(pub);
        TRACE(t == 0, it, 4);

        // ---- global stores that need nothing from the other warps: the y-edge and corner exports ----
        if (row_lo || row_hi) {                                            // the row beyond the tile edge receives exactly Um (Up)
            if (store_rho) (ro.y + k * ro.s_y)[zt * psy + ((row_lo ? btym : btyp) * 2 + (row_lo ? 1 : 0)) * nx + x] = row_lo ? pm : pp;
        }

        TRACE(t == 0, it, 5);
        mbar_wait(pub, it & 1);
        TRACE(t == 0, it, 6);

        // ---- y stage of the gather; exports across the tile's x edges ----
        {
            T out = p0;
            if (!row_lo) out += SUup[own_s - RW];                          // Up(y-1)
            if (!row_hi) out += SUum[own_s + RW];                          // Um(y+1)
            if (store_rho) ro_in[(long long)zt * pl] = out;
            if (lane_lo || lane_hi) {
                const int vc = lane_lo ? own_s - 1 : own_s + 1;            // the virtual column next to this lane
                T a_0 = ee[1];
                if (!row_lo) a_0 += SUup[vc - RW];
                if (!row_hi) a_0 += SUum[vc + RW];
                const T hout = col_acc[0] + ee[0];
                col_acc[0] = col_acc[1] + a_0;
                col_acc[1] = ee[2];
                if (store_rho) (ro.x + k * ro.s_x)[zt * psx + ((bty * ntx + (lane_lo ? btxm : btxp)) * 2 + (lane_lo ? 1 : 0)) * TY + ty] = hout;
            }
        }
        zt = zl;
        zl = zl + 1 == nz ? 0 : zl + 1;
        if (HAS_SOLID && it + 1 < niter) lk = __ldg(links + (long long)zl * pl + own_xy);
    }
}

}  // namespace lb
