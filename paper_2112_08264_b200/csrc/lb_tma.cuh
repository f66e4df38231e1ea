// lb_tma.cuh -- the fused one-pass time step with TMA-staged populations (the hot kernel on B200).
//
// Same algorithm and same state convention as lb_onepass.cuh (h-state, pull streaming, density carried
// from step to step through the four single-writer arrays rho_in / rho_x / rho_y / rho_xy), but the
// 38 population planes of a tile are brought into shared memory by the TMA unit instead of by 38
// per-thread loads, and one thread handles one (node, component) instead of one node:
//   * one producer warp per CTA issues, per z plane, 19 `cp.async.bulk.tensor.4d` box loads (one per
//     direction; the box spans the two adjacent planes of the two components, pop_plane(); box = tile
//     shifted by -c_i in y and z) that complete on an mbarrier; the consumer threads then read their 19
//     values with LDS at fixed offsets: no per-thread address arithmetic, no registers in flight, and the
//     prefetch distance is a whole plane whatever the occupancy is;
//   * measured on B200: a TMA box whose innermost start is not 16-byte aligned
//     raises an illegal-instruction fault, so the x shift cannot be given to the TMA.  Directions with
//     c_x != 0 are loaded as an ALIGNED box that is PADX = 16/sizeof(T) elements wider, and the consumer
//     applies the shift in its LDS address (free);
//   * the TMA zero-fills out-of-range box parts and does not wrap.  x: tiles at the box
//     boundary load, per direction with c_x != 0, one more box (PADX x TY) holding the wrapped column,
//     and the lane next to the edge reads that box instead (a different base offset, same instruction).
//     y: the one warp whose row lies beyond the edge re-loads its 5 affected populations with plain loads.
//     z wraps in the box coordinate;
//   * two shared-memory stages: consumers copy their plane into registers and release its stage at once, and the
//     producer sends for plane j as soon as every consumer warp has left plane j - 2, two iterations before
//     its use: the loads come straight from DRAM, no L2 prefetch; post-collision values are stored straight
//     from registers (aligned, coalesced);
//   * the two threads of a node exchange rho^k, j^k (common velocity, S4) through stage entries they have
//     already consumed, with a 64-thread named barrier per tile row; the y stage of the density gather is
//     double-buffered behind one mbarrier per (row, component): a warp waits only for the rows above and
//     below it (arrive, independent stores, wait); the stage hand-off is mbarriers only;
//   * three more warps of the producer group assemble the density ring one plane per iteration: every ring
//     thread owns up to four ring positions for the whole kernel (their piece offsets are tabulated in shared
//     memory), fetches their pieces with cp.async one iteration ahead and adds them up in the fixed order; a
//     thread only ever reads landing slots it filled itself, so the ring warps need no barrier among themselves;
//   * the producer warp group hands registers to the consumers (setmaxnreg): 16 consumer warps at 112
//     registers, producer group at 32;
//   * optional fused diagnostics (DIAG): per plane a four-value warp reduction of the post-collision moments.
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
// both barriers have completed the phase of the given parity
__device__ __forceinline__ void mbar_wait2(void* bar_a, void* bar_b, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred PA, PB;\n\tLAB_WAIT2:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 PA, [%0], %2, 0x989680;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 PB, [%1], %2, 0x989680;\n\t"
        "and.pred PA, PA, PB;\n\t"
        "@!PA bra LAB_WAIT2;\n\t}" ::"r"(smem_u32(bar_a)), "r"(smem_u32(bar_b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_wait3(void* bar_a, void* bar_b, void* bar_c, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred PA, PB, PC;\n\tLAB_WAIT3:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 PA, [%0], %3, 0x989680;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 PB, [%1], %3, 0x989680;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 PC, [%2], %3, 0x989680;\n\t"
        "and.pred PA, PA, PB;\n\t"
        "and.pred PA, PA, PC;\n\t"
        "@!PA bra LAB_WAIT3;\n\t}" ::"r"(smem_u32(bar_a)), "r"(smem_u32(bar_b)), "r"(smem_u32(bar_c)), "r"(parity) : "memory");
}
// box load: coordinates (x, y, z, plane); x * sizeof(T) must be a multiple of 16 (see header)
// `pol`: an L2 eviction policy (l2_policy_*)
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, void* bar, int c0, int c1, int c2, int c3, unsigned long long pol) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6}], [%2], %7;"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol) : "memory");
}
// plain global stores through a pointer the compiler must treat as opaque (see the running store pointer in the kernel)
// Streaming (.cs: evict-first in L2): a stored population is next read one time step later, when L2 has long turned over, while
// the lines the TMA reads are wanted once more by the tile next door (the 16-byte margins of the wide boxes): with the stores
// evict-first and the loads evict-last more of those second reads hit (512^3 fp64 in bench.py: 16.1 -> 15.9 ms per step).
__device__ __forceinline__ void st_global(double* p, double v) { asm volatile("st.global.cs.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }
__device__ __forceinline__ void st_global(float* p, float v) { asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }
__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
    unsigned long long p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
    unsigned long long p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_normal() {
    unsigned long long p; asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p)); return p;
}
// p += step16 * 16 bytes in ONE instruction (IMAD.WIDE.U32 on the otherwise idle fp32/integer-multiply pipe) instead of
// the add-with-carry pair the compiler emits for a 64-bit pointer increment
template <typename T>
__device__ __forceinline__ void ptr_step16(T*& p, unsigned step16) { asm volatile("mad.wide.u32 %0, %1, 16, %0;" : "+l"(p) : "r"(step16)); }
// products and sums the compiler may not contract into an fma
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }

// ---- shared-memory layout -----------------------------------------------------------------------------
template <typename T, int TY>
struct TmaLayout {
    static constexpr int TX = 32, NT = TX * TY;
    static constexpr int PADX = 16 / int(sizeof(T));                   // elements per 16 bytes
    static constexpr int W = TX + PADX;                                // row length of a wide (c_x != 0) box
    static constexpr int RW = TX + 2, RH = TY + 2, RS = RW * RH;       // density ring plane: tile + one-node frame
    static constexpr int SUP = TY * RW;                                // one y-stage plane: tile rows with an x frame
    // one stage slot per direction, both components in it (the box spans their two planes): [k][TY][TX] (c_x = 0) or
    // [k][TY][W] followed by the wrapped-column box [k][TY][PADX] (c_x != 0).  TMA destinations are 128-byte aligned.
    static constexpr int NA = 2 * NT;                                  // narrow slot
    static constexpr int XC = 2 * W * TY;                              // offset of the wrapped-column box inside a wide slot
    static constexpr int WA = XC + 2 * PADX * TY;                      // wide slot
    static_assert((NA * sizeof(T)) % 128 == 0 && (XC * sizeof(T)) % 128 == 0 && (WA * sizeof(T)) % 128 == 0, "TMA destination alignment");
    // number of wide slots before direction i (the directions with c_x != 0 are 1, 2, 7..14)
    __host__ __device__ static constexpr int wide_before(int i) { return (i > 1) + (i > 2) + (i > 7 ? (i - 7 < 8 ? i - 7 : 8) : 0); }
    __host__ __device__ static constexpr int slot_off(int i) { return (i - wide_before(i)) * NA + wide_before(i) * WA; }
    static constexpr int STAGE_ELEMS = slot_off(Q);                    // one stage: the 19 slots of one z plane
    static constexpr unsigned STAGE_TX_BYTES = unsigned(2 * (9 * NT + 10 * W * TY) * sizeof(T));   // bytes the 19 boxes deliver
    static constexpr unsigned XCOL_TX_BYTES = unsigned(2 * 5 * PADX * TY * sizeof(T));             // ... plus the 5 wrapped-column boxes of one x side
    static constexpr int STAGE = 0;                                    // [2][STAGE_ELEMS] two stages: plane `it` lives in stage it & 1
    static constexpr int RING = STAGE + 2 * STAGE_ELEMS;               // [4][2][RS]      rho(t), planes z-1..z+2
    static constexpr int SU = RING + 8 * RS;                           // [2][2][2][SUP]  double-buffered z-summed Up, Um per component
    static constexpr int LAND = SU + 8 * SUP;                          // [2][8][96]      landing slots of the ring pieces, per component and ring thread
    static constexpr int EX = LAND + 2 * 8 * 96;                           // [2 TY][2][8]    per tile row and x side: what leaves the tile in x by c_z, and the z pipeline of that export
    static constexpr int CST = EX + 2 * TY * 2 * 8;                    // {om_r, om_b, G, sigma, beta, 1/nu_r, 1/nu_b}
    static constexpr int RTAB = CST + 10;                              // CST + 8: int {iterations of this CTA, its first plane}                               // int [9][96]     where the ring threads' pieces live
    static constexpr int END = RTAB + (9 * 96 * int(sizeof(int)) + int(sizeof(T)) - 1) / int(sizeof(T));
    static constexpr size_t BAR_BYTE_OFF = (size_t(END) * sizeof(T) + 15) / 16 * 16;
    // mbarriers: full[2], done[2], rdy, rowpub[2][2 TY]
    static constexpr int NBARS = 5 + 4 * TY;
    static constexpr size_t WACC_BYTE_OFF = BAR_BYTE_OFF + NBARS * sizeof(unsigned long long);   // double [2 TY][4]: per-warp sums (DIAG)
    static constexpr size_t BYTES = WACC_BYTE_OFF + 2 * TY * 4 * sizeof(double);
    static_assert(BYTES <= 227 * 1024, "shared memory per CTA");
};



// ---- which z chunk a CTA takes ---------------------------------------------------------------------------------
// Grid (ntx, nty, chunks).  Tile columns col = bty ntx + btx < col_split are cut into nz / zc chunks of zc planes; the columns from
// col_split on (the host picks how many, so that the number of working CTAs is a multiple of the SM count: one CTA per SM, and a
// last wave that leaves a third of the SMs idle costs more than it looks) into one chunk more, of nz / (nz / zc + 1) planes or one
// more; the grid then has one more z layer, in which only those columns work.  Returns false for a CTA without work; niter =
// planes + 2.
__device__ __forceinline__ bool chunk_range(int col, int col_split, int nz, int zc, int& z0, int& niter) {
    const int c = blockIdx.z;
    if (col < col_split) {
        if (c * zc >= nz) return false;
        z0 = c * zc;
        niter = zc + 2;
    } else {
        const int m = nz / zc + 1;
        z0 = c * nz / m;
        niter = (c + 1) * nz / m - z0 + 2;
    }
    return true;
}

// ---- the kernel ------------------------------------------------------------------------------------------
// Threads: 2*NT consumers (component k = t / NT, node (tx, ty) = ((t % NT) % 32, (t % NT) / 32): one warp per
// tile row and component) followed by one producer warp group (TMA warp + 3 ring warps).  The producer
// group gives its registers to the consumers (setmaxnreg), which is why it is a whole warp group.
// DIAG (boxes without solids): the kernel also leaves the per-component mass and the total momentum of the state AFTER this step
// behind, one partial per CTA: the post-collision moments sum_i f*_i = rho, sum_i f*_i c_i = (1 - om) j + om rho u' + rho du
// (Eq. 1, Eq. 10, S5), which streaming in a periodic box only permutes.  Per plane a four-value warp reduction (6 shuffles of
// doubles) into per-warp shared-memory sums; at the end the 2 TY warp sums in a fixed order.
// MODEL 1 (boxes without solids): the colour-gradient collision instead of Shan-Chen force + BGK.  The ring
// then holds the phase field Theta of the tile and its frame (the ring warps turn the two assembled densities into Theta), a
// thread reads BOTH components' populations of its node from the stage (the recolouring works on their sum) and computes its own
// component's post-collision values: the two threads of a node need no exchange.  G carries sigma, the extra parameter beta.
template <typename T, bool HAS_SOLID, int TY, bool DIAG = false, int MODEL = 0>
__global__ void __launch_bounds__(2 * 32 * TY + 128, 1)
k_step_tma(const __grid_constant__ CUtensorMap tm_n, const __grid_constant__ CUtensorMap tm_w,
           const __grid_constant__ CUtensorMap tm_c, const T* __restrict__ h, T* __restrict__ g, const unsigned* __restrict__ links,
           const RhoView<T> ri, const RhoView<T> ro, long long NP, int nx, int ny, int nz, int zc,
           T om_r, T om_b, T G, double* __restrict__ diag_part = nullptr, T beta = T(0), int col_split = 1 << 30) {
    static_assert(!(DIAG && HAS_SOLID), "the fused sums assume periodic streaming without bounce-back");
    static_assert(!(MODEL != 0 && (HAS_SOLID || DIAG)), "the colour-gradient variant is built for boxes without solids, without fused sums");
    using L = TmaLayout<T, TY>;
    constexpr int TX = L::TX, NT = L::NT, NC = 2 * NT, RW = L::RW, RS = L::RS, SUP = L::SUP, W = L::W, PADX = L::PADX;
    static_assert(TY >= 2 && TY <= 8, "one named barrier per tile row (ids 1..TY)");
    // register hand-over between the warp groups: (2*NT + 128) threads start with 65536 / threads registers each
    constexpr int START_REGS = (65536 / (NC + 128)) / 8 * 8;
    constexpr int PRODUCER_REGS = 32;
    constexpr int CONSUMER_REGS = (START_REGS + (START_REGS - PRODUCER_REGS) * 128 / NC) / 8 * 8;
    extern __shared__ __align__(1024) unsigned char smem_tma[];
    T* sm = reinterpret_cast<T*>(smem_tma);
    T* stage = sm + L::STAGE;
    T* ring = sm + L::RING;
    T* SUb = sm + L::SU;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_tma + L::BAR_BYTE_OFF);
    unsigned long long* full = bars;          // [2] the 19 boxes of plane `it` have landed in stage it & 1 (tx bytes)
    unsigned long long* done = bars + 2;      // [2] every consumer warp has taken what it needs out of stage it & 1
    unsigned long long* rdy = bars + 4;       // the ring warps have assembled the density ring plane this iteration needs
    unsigned long long* rowpub = bars + 5;    // [2][2 TY] warp (k, ty) has published its y-stage inputs of plane `it`: rowpub[it & 1][k TY + ty]

    const int t = threadIdx.x;
    const int ntx = nx / TX, nty = ny / TY;
    const int btx = blockIdx.x, bty = blockIdx.y;
    const int x0 = btx * TX, y0 = bty * TY;
    int z0, niter_cta;                        // planes z0-1 .. z0+niter-2; the first and the last are re-collided only
    if (!chunk_range(bty * ntx + btx, col_split, nz, zc, z0, niter_cta)) return;   // (the host guarantees nz % zc == 0)
    // The iteration count differs between CTAs: it lives in shared memory and is re-read where it is used (a register held across
    // the plane loop costs the consumers a spill: +9 local loads per plane, 3.5 % of the step).
    int* const niter_slot = reinterpret_cast<int*>(sm + L::CST + 8);
    auto NITER = [&]() { return *reinterpret_cast<volatile const int*>(niter_slot); };
    auto Z0 = [&]() { return *reinterpret_cast<volatile const int*>(niter_slot + 1); };   // likewise, for the producer group (32 registers)
    const long long pl = (long long)nx * ny;
    const bool wrap_xlo = btx == 0, wrap_xhi = btx == ntx - 1;             // the TMA zero-fills outside the box: x wraps with an
                                                                           // extra box per direction, y with consumer loads
    auto wrapz = [&](int p) { p %= nz; return p < 0 ? p + nz : p; };

    if (t == 0) {
        niter_slot[0] = niter_cta; niter_slot[1] = z0;
        for (int s = 0; s < 2; ++s) { mbar_init(full + s, 1); mbar_init(done + s, 2 * TY); }
        mbar_init(rdy, 3);
        for (int b = 0; b < 4 * TY; ++b) mbar_init(rowpub + b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        sm[L::CST + 0] = om_r; sm[L::CST + 1] = om_b; sm[L::CST + 2] = G; sm[L::CST + 3] = G; sm[L::CST + 4] = beta;
        sm[L::CST + 5] = T(3) / (T(1) / om_r - T(0.5)); sm[L::CST + 6] = T(3) / (T(1) / om_b - T(0.5));   // 1 / nu_k, nu_k = c_s^2 (tau_k - 1/2)
    }
    __syncthreads();

    // =================================== producer warp group ===================================
    if (t >= NC) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
        if (t >= NC + 32) {
            // ---- ring warps (3): the density ring, one plane per iteration, two planes ahead of its use.  Ring position
            //      pos (tile + one-node frame) of either component is the sum ((in + x) + y) + xy of up to four single-writer
            //      pieces (lb_onepass.cuh).  Thread r owns positions r, r + 96, ... (at most NPOS = 4) with, for this geometry,
            //      at most one x piece, two y pieces and one xy piece among them: it fetches those pieces itself (cp.async, one
            //      iteration ahead) and only ever reads landing slots it filled itself, so the ring warps need no barrier among
            //      themselves.  Where the pieces live is tabulated once, in shared memory (these warps run on 32 registers):
            //      rt[j][r], j = 0..3 the `in` pieces, 4 the x piece, 5 and 6 the y pieces, 7 the xy piece (element offsets
            //      inside one z plane of their arrays, -1 = none), 8 the positions the extra pieces belong to (2 bits each). ----
            const int r = t - NC - 32;
            constexpr int NR = 96, NPOS = (RS + NR - 1) / NR;
            static_assert(NPOS == 4, "ring table layout");
            int* rt = reinterpret_cast<int*>(sm + L::RTAB) + r;
            {
                int ox = -1, oya = -1, oyb = -1, oxy = -1, who = 0;
#pragma unroll 1
                for (int m = 0; m < NPOS; ++m) {
                    const int pos = r + m * NR;
                    int oin = -1;
                    if (pos < RS) {
                        const int rx = pos % RW - 1, ry = pos / RW - 1;
                        const int txm = btx == 0 ? ntx - 1 : btx - 1, txp = btx == ntx - 1 ? 0 : btx + 1;
                        const int tym = bty == 0 ? nty - 1 : bty - 1, typ = bty == nty - 1 ? 0 : bty + 1;
                        const int otx = rx < 0 ? txm : (rx >= TX ? txp : btx), oty = ry < 0 ? tym : (ry >= TY ? typ : bty);
                        const int lx = rx < 0 ? TX - 1 : (rx >= TX ? 0 : rx), ly = ry < 0 ? TY - 1 : (ry >= TY ? 0 : ry);
                        const bool xe = lx == 0 || lx == TX - 1, ye = ly == 0 || ly == TY - 1;   // edge column / row of its owner tile
                        oin = (oty * TY + ly) * nx + otx * TX + lx;
                        if (xe) {
                            if (ox >= 0) __trap();                         // geometry: one x piece per thread
                            ox = ((oty * ntx + otx) * 2 + (lx != 0)) * TY + ly; who |= m;
                        }
                        if (ye) {
                            const int oy = (oty * 2 + (ly != 0)) * nx + otx * TX + lx;
                            if (oya < 0) { oya = oy; who |= m << 2; }
                            else if (oyb < 0) { oyb = oy; who |= m << 4; }
                            else __trap();                                 // geometry: two y pieces per thread
                        }
                        if (xe && ye) {
                            if (oxy >= 0) __trap();
                            oxy = (oty * ntx + otx) * 4 + (ly != 0) * 2 + (lx != 0); who |= m << 6;
                        }
                    }
                    rt[m * NR] = oin;
                }
                rt[4 * NR] = ox; rt[5 * NR] = oya; rt[6 * NR] = oyb; rt[7 * NR] = oxy; rt[8 * NR] = who;
            }
            const unsigned psx_ = unsigned(nty * ntx * 2 * TY), psy_ = unsigned(nty * 2 * nx), psxy_ = unsigned(nty * ntx * 4);
            T* land = sm + L::LAND + r;                                    // [2][8][96]: per component the 4 `in`, x, y, y, xy landing slots of thread r
            // ask for the pieces of ring plane rp (= box plane z0 - 2 + rp): asynchronous, no registers in flight
            auto ring_fetch = [&](int rp) {
                const unsigned zp = unsigned(wrapz(Z0() - 2 + rp));
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int off = rt[j * NR];
                    if (off >= 0) {
                        const T* b0 = j < 4 ? ri.in : (j == 4 ? ri.x : (j < 7 ? ri.y : ri.xy));
                        const long long cs = j < 4 ? ri.s_in : (j == 4 ? ri.s_x : (j < 7 ? ri.s_y : ri.s_xy));
                        const unsigned ps = j < 4 ? unsigned(pl) : (j == 4 ? psx_ : (j < 7 ? psy_ : psxy_));
                        const T* src = b0 + (zp * ps + unsigned(off));
                        cp_async<sizeof(T)>(land + j * NR, src);
                        cp_async<sizeof(T)>(land + (8 + j) * NR, src + cs);
                    }
                }
                cp_async_commit();
            };
            // ... and add them up in the fixed order ((in + x) + y) + xy once they have landed (own copies only)
            auto ring_assemble = [&](int rp) {
                cp_async_wait<0>();
                T* dst = ring + (rp & 3) * 2 * RS + r;
                const int who = rt[8 * NR];
                const bool hx = rt[4 * NR] >= 0, hya = rt[5 * NR] >= 0, hyb = rt[6 * NR] >= 0, hxy = rt[7 * NR] >= 0;
                const int mx = who & 3, mya = (who >> 2) & 3, myb = (who >> 4) & 3, mxy = (who >> 6) & 3;
#pragma unroll
                for (int kk = 0; kk < 2; ++kk) {
                    const T* ld = land + kk * 8 * NR;
                    T v[NPOS];
#pragma unroll
                    for (int m = 0; m < NPOS; ++m) v[m] = ld[m * NR];
                    const T px = ld[4 * NR], pya = ld[5 * NR], pyb = ld[6 * NR], pxy = ld[7 * NR];
#pragma unroll
                    for (int m = 0; m < NPOS; ++m) {
                        if (hx && mx == m) v[m] += px;
                        if (hya && mya == m) v[m] += pya;
                        if (hyb && myb == m) v[m] += pyb;
                        if (hxy && mxy == m) v[m] += pxy;
                        if (m < NPOS - 1 || r + m * NR < RS) dst[kk * RS + m * NR] = v[m];
                    }
                }
                if (MODEL == 1) {                                           // Theta = (rho^1 - rho^2) / (rho^1 + rho^2), 0 where empty
#pragma unroll
                    for (int m = 0; m < NPOS; ++m)
                        if (m < NPOS - 1 || r + m * NR < RS) {
                            const T a = dst[m * NR], b = dst[RS + m * NR], sum = a + b;
                            dst[m * NR] = sum != T(0) ? (a - b) / sum : T(0);
                        }
                }
            };
            for (int rp = 0; rp < 2; ++rp) {                                // iteration 0 needs ring planes 0, 1, 2
                ring_fetch(rp);
                ring_assemble(rp);
            }
            ring_fetch(2);
            for (int j = 0; j < NITER(); ++j) {
                // ring plane j+2 (the z+1 neighbour plane of iteration j): its slot held plane j-2, last read in iteration
                // j-2, which every consumer warp had left when it arrived on done(j-1)
                if (j > 0) mbar_wait(done + ((j - 1) & 1), ((j - 1) >> 1) & 1);
                ring_assemble(j + 2);
                __syncwarp();
                if ((r & 31) == 0) mbar_arrive(rdy);
                if (j + 3 <= NITER() + 1) ring_fetch(j + 3);
            }
            return;
        }
        // ---- TMA warp: plane j goes into stage j & 1 as soon as every consumer warp has left plane j - 2: a whole iteration
        //      ahead of its use, so the loads come straight from DRAM and need no L2 prefetch ----
        const int lane = t - NC;
#ifndef LB_POL_N
#define LB_POL_N l2_policy_evict_last
#define LB_POL_W l2_policy_evict_last
#endif
        const unsigned long long pol_n = LB_POL_N(), pol_w = LB_POL_W();
        for (int j = 0; j < NITER(); ++j) {
            const int z = Z0() - 1 + j;
            const int zw[3] = {wrapz(z - 1), wrapz(z), wrapz(z + 1)};
            if (lane == 0) {
                const int s = j & 1;
                if (j >= 2) mbar_wait(done + s, ((j >> 1) - 1) & 1);
                mbar_expect_tx(full + s, L::STAGE_TX_BYTES + (wrap_xlo ? L::XCOL_TX_BYTES : 0u) + (wrap_xhi ? L::XCOL_TX_BYTES : 0u));
#pragma unroll
                for (int i = 0; i < Q; ++i) {
                    const int zq = zw[1 - dir_cz(i)];                       // f_i(x) = h_i(x - c_i)
                    const int q = pop_plane(0, i);                          // the box takes planes q, q + 1: both components
                    T* slot = stage + s * L::STAGE_ELEMS + L::slot_off(i);
                    if (dir_cx(i) == 0) tma_load_4d(slot, &tm_n, full + s, x0, y0 - dir_cy(i), zq, q, pol_n);
                    else {
                        tma_load_4d(slot, &tm_w, full + s, dir_cx(i) > 0 ? x0 - PADX : x0, y0 - dir_cy(i), zq, q, pol_w);
                        // the column beyond the box edge: columns nx-PADX..nx-1 for c_x > 0, 0..PADX-1 for c_x < 0
                        if (dir_cx(i) > 0 && wrap_xlo) tma_load_4d(slot + L::XC, &tm_c, full + s, nx - PADX, y0 - dir_cy(i), zq, q, pol_w);
                        if (dir_cx(i) < 0 && wrap_xhi) tma_load_4d(slot + L::XC, &tm_c, full + s, 0, y0 - dir_cy(i), zq, q, pol_w);
                    }
                }
            }
            __syncwarp();
        }
        return;
    }

    // =================================== consumers ===================================
    // Register diet: with 227 KB of shared memory there is no L1 left, so a spilled register is an L2 round trip (measured:
    // ~400 cycles per reload).  Whatever is only needed now and then lives elsewhere: global addresses are 32-bit element
    // offsets added to the kernel parameters at the point of use, om / G are re-read from shared memory, and the state of
    // the x-edge exports (two lanes per warp) lives in shared memory instead of in every lane's registers.
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
    const int k = t / NT;                                                  // component of this thread (warp-uniform)
    const int tl = t - k * NT;
    const int tx = tl % TX, ty = tl / TX;
    const bool lane_lo = tx == 0, lane_hi = tx == TX - 1, row_lo = ty == 0, row_hi = ty == TY - 1;
    const int own_r = (ty + 1) * RW + tx + 1;                              // ring position (tile + frame); the y-stage planes have no frame rows: own_r - RW
    const T zero = T(0);
    const T omc = T(1) - (k == 0 ? om_r : om_b);
    // element offsets of this thread's targets inside one z plane of the arrays (component included); + z * plane stride
    const unsigned e_own = unsigned((long long)k * NP + (long long)(y0 + ty) * nx + x0 + tx);   // populations (plane pop_plane(k, 0) = k) and rho_in (s_in == NP)
    // the export targets across the tile's x edge / y edge / corner are computed where they are used (few lanes, once per
    // plane) from these CTA-uniform tile indices; `opaque` keeps the compiler from hoisting them into registers for the whole loop
    const int btxm = btx == 0 ? ntx - 1 : btx - 1, btxp = btx == ntx - 1 ? 0 : btx + 1;
    const int btym = bty == 0 ? nty - 1 : bty - 1, btyp = bty == nty - 1 ? 0 : bty + 1;
    auto opaque = [](int v) { asm volatile("" : "+r"(v)); return v; };
    const unsigned psx = unsigned(nty * ntx * 2 * TY), psy = unsigned(nty * 2 * nx), psxy = unsigned(nty * ntx * 4), plu = unsigned(pl);
    const unsigned step16 = unsigned((2 * NP * (long long)sizeof(T)) >> 4);   // two planes, in 16-byte units (NP is a multiple of 64)
    const T* ring_o = ring + (1 - k) * RS + own_r;                         // the OTHER component's density (S2), at this node
    T* SUk = SUb + k * 2 * SUP + own_r - RW;                               // this node in the y-stage planes (x frame only)
    T* exs = sm + L::EX + ((k * TY + ty) * 2 + (lane_hi ? 1 : 0)) * 8;     // edge lanes: {ee[0..2], col_acc[0..1]} of this row and side
    const volatile T* cst = sm + L::CST;                                   // {om_r, om_b, G}
    // where this thread finds f_i = h_i(x - c_i) inside slot i, by c_x: the x shift is applied here; the lane next to the
    // box edge reads the wrapped-column box instead
    const int rd0 = k * NT + ty * TX + tx;
    const int rdp = (wrap_xlo && lane_lo) ? L::XC + (k * TY + ty) * PADX + PADX - 1 : (k * TY + ty) * W + tx + PADX - 1;
    const int rdm = (wrap_xhi && lane_hi) ? L::XC + (k * TY + ty) * PADX : (k * TY + ty) * W + tx + 1;
    const bool wrap_ylo = bty == 0 && row_lo, wrap_yhi = bty == nty - 1 && row_hi;   // warp-uniform
    if (lane_lo || lane_hi) { exs[3] = zero; exs[4] = zero; }

    // ---- per-thread state carried along z ----
    // z pipelines of the density gather (see the collision below)
    T qa0 = zero, qb0 = zero, qap = zero, qbp = zero, qam = zero, qbm = zero;

    int zl = wrapz(z0 - 1), zt = wrapz(z0 - 2);         // this plane / the plane the gathered density belongs to
    unsigned lk = 0;
    if (HAS_SOLID) lk = __ldg(links + (e_own - unsigned(k * NP)) + (long long)zl * pl);

#pragma unroll 1
    for (int it = 0; it < NITER(); ++it) {
        const bool store_h = it >= 1 && it <= NITER() - 2;
        const bool store_rho = it >= 2;                 // target plane z-1 lies in [z0, z1)
        const int s0 = (it + 1) & 3;                    // ring slot of plane z
        const bool fluid = !HAS_SOLID || !(lk & OP_SOLID_BIT);   // nothing happens inside a particle
        const int sg = it & 1;                          // stage of this plane
        const unsigned ph = (it >> 1) & 1;              // phase parity of the alternating barriers
        T* st = stage + sg * L::STAGE_ELEMS;
        T* SU = SUk + sg * 4 * SUP;

        // ---- pull: the stage holds h_i(x - c_i) for the whole tile (Eq. 5, periodic) ----
        mbar_wait(full + sg, ph);
        mbar_wait(rdy, it & 1);                         // density ring planes z-1, z, z+1 are in place (before `done`: the ring
                                                        // warps must not get two phases ahead of any waiter)
        T f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = st[L::slot_off(i) + (dir_cx(i) == 0 ? rd0 : (dir_cx(i) > 0 ? rdp : rdm))];
        if (wrap_ylo || wrap_yhi) {                     // the row beyond the box edge in y (one warp of a boundary tile): plain loads
            const int gy = wrap_ylo ? ny - 1 : 0;
            const int x = x0 + tx;
            const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
            const long long zs[3] = {(long long)zt * pl, (long long)zl * pl, (long long)(zl + 1 == nz ? 0 : zl + 1) * pl};
#pragma unroll
            for (int i = 1; i < Q; ++i)
                if (dir_cy(i) != 0) {
                    const T v = __ldg(h + (long long)pop_plane(k, i) * NP + zs[1 - dir_cz(i)] + (long long)gy * nx + xs[1 - dir_cx(i)]);
                    if ((dir_cy(i) > 0 && wrap_ylo) || (dir_cy(i) < 0 && wrap_yhi)) f[i] = v;
                }
        }
        if (HAS_SOLID && (lk & 0x7FFFEu)) {             // halfway bounce-back (Eq. 23-24, u_b = 0): f_i(x) = h_opp(i)(x) when x - c_i is solid
            const T* hn = h + (e_own + zl * plu);
#pragma unroll
            for (int i = 1; i < Q; ++i)
                if (lk >> dir_opp(i) & 1u) f[i] = __ldg(hn + (long long)(2 * dir_opp(i)) * NP);
        }

        T rho = zero, jx = zero, jy = zero, jz = zero;
        T ux = zero, uy = zero, uz = zero, ex = zero, ey = zero, ez = zero;
        T cg_rt = zero, cg_x = zero, cg_om = zero, cg_amp = zero, cg_ig2 = zero, cg_ign = zero, cg_rcs = zero;   // MODEL 1 (ex, ey, ez then hold grad Theta)
        if constexpr (MODEL == 1) {
            // ---- colour gradient: the other component's populations of this node come out of the same stage; f becomes the colour-blind
            //      sum, the two densities are summed on the way in the order of moments19 ----
            const int dk = 1 - 2 * k;
            const int od0 = dk * NT;
            const int odp = dk * ((wrap_xlo && lane_lo) ? TY * PADX : TY * W), odm = dk * ((wrap_xhi && lane_hi) ? TY * PADX : TY * W);
            T fo[Q];
#pragma unroll
            for (int i = 0; i < Q; ++i) fo[i] = st[L::slot_off(i) + (dir_cx(i) == 0 ? rd0 + od0 : (dir_cx(i) > 0 ? rdp + odp : rdm + odm))];
            if (wrap_ylo || wrap_yhi) {
                const int gy = wrap_ylo ? ny - 1 : 0;
                const int x = x0 + tx;
                const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
                const long long zs[3] = {(long long)zt * pl, (long long)zl * pl, (long long)(zl + 1 == nz ? 0 : zl + 1) * pl};
#pragma unroll
                for (int i = 1; i < Q; ++i)
                    if (dir_cy(i) != 0) {
                        const T v = __ldg(h + (long long)pop_plane(1 - k, i) * NP + zs[1 - dir_cz(i)] + (long long)gy * nx + xs[1 - dir_cx(i)]);
                        if ((dir_cy(i) > 0 && wrap_ylo) || (dir_cy(i) < 0 && wrap_yhi)) fo[i] = v;
                    }
            }
            T r_own = f[0], r_oth = fo[0];
            f[0] += fo[0];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                r_own += f[2 * p + 1] + f[2 * p + 2];
                r_oth += fo[2 * p + 1] + fo[2 * p + 2];
                f[2 * p + 1] += fo[2 * p + 1]; f[2 * p + 2] += fo[2 * p + 2];
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy reads of the stage before the TMA's next writes
            __syncwarp();
            if (lane_lo) mbar_arrive(done + sg);        // the producer may refill this stage with the plane after next
            moments19<T>(f, cg_rt, jx, jy, jz);         // rho and rho u of the mixture (Eq. 7)
            if (cg_rt != zero) {
                const T irt = T(1) / cg_rt;
                ux = jx * irt; uy = jy * irt; uz = jz * irt;
                cg_x = r_own * irt;
                const T x_oth = r_oth * irt;
                const T inv_nu = cg_x * cst[5 + k] + x_oth * cst[6 - k];                            // 1 / nu
                cg_om = T(2) / (T(6) / inv_nu + T(1));                                             // reading C2
                // grad Theta = (1 / c_s^2) sum_i w_i Theta(x + c_i) c_i from the ring (reading C1)
                const T* ring_t = ring + own_r;
                T d[9];
#pragma unroll
                for (int p = 0; p < 9; ++p) {
                    const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                    d[p] = w_pair<T>(p) * (ring_t[sp * 2 * RS + pair_cy(p) * RW + pair_cx(p)] - ring_t[sm_ * 2 * RS - pair_cy(p) * RW - pair_cx(p)]);
                }
                ex = T(3) * ((((d[0] + d[3]) + d[4]) + d[5]) + d[6]);
                ey = T(3) * ((((d[1] + d[3]) - d[4]) + d[7]) + d[8]);
                ez = T(3) * ((((d[2] + d[5]) - d[6]) + d[7]) - d[8]);
                const T g2 = ex * ex + ey * ey + ez * ez;
                if (g2 != zero) { cg_ig2 = T(1) / g2; cg_ign = T(1) / sqrt(g2); }
                cg_amp = T(0.5) * (T(2.25) * cst[3] * cg_om) * (g2 * cg_ign);                      // (A / 2) |grad|, A = (9/4) sigma omega (Eq. 19)
                cg_rcs = (k == 0 ? cst[4] : -cst[4]) * cg_x * x_oth * cg_rt;                       // +- beta rho^1 rho^2 / rho
            }
        }
        if constexpr (MODEL == 0) {
        // ---- moments of this component (Eq. 6-7), exchanged with the other component's thread of the same node ----
        if (fluid) moments19<T>(f, rho, jx, jy, jz);
        else {
#pragma unroll
            for (int i = 0; i < Q; ++i) f[i] = zero;
        }
        // The partner's moments.  fp64 (and with solids): exchanged through stage elements this thread has just consumed (its own
        // entries of four c_x = 0 slots; the stage is only refilled after `done`, on which a warp arrives after it has read its
        // partner's values), behind a named barrier of the two warps of the tile row.  fp32 without solids: each thread sums the
        // partner's 19 populations out of the stage itself (same order, so both threads get the same bits): 19 LDS + 45 adds are
        // cheaper there than the barrier (measured at 512^3: fp32 8.95 -> 8.80 ms; fp64 15.4 -> 15.7 ms, so fp64 keeps the exchange).
        constexpr bool XCHG = sizeof(T) == 8 || HAS_SOLID;
        T orho, ojx, ojy, ojz;
        if constexpr (!XCHG) {
            const int dk = 1 - 2 * k;
            const int od0 = dk * NT;
            const int odp = dk * ((wrap_xlo && lane_lo) ? TY * PADX : TY * W), odm = dk * ((wrap_xhi && lane_hi) ? TY * PADX : TY * W);
            T fo[Q];
#pragma unroll
            for (int i = 0; i < Q; ++i) fo[i] = st[L::slot_off(i) + (dir_cx(i) == 0 ? rd0 + od0 : (dir_cx(i) > 0 ? rdp + odp : rdm + odm))];
            if (wrap_ylo || wrap_yhi) {
                const int gy = wrap_ylo ? ny - 1 : 0;
                const int x = x0 + tx;
                const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
                const long long zs[3] = {(long long)zt * pl, (long long)zl * pl, (long long)(zl + 1 == nz ? 0 : zl + 1) * pl};
#pragma unroll
                for (int i = 1; i < Q; ++i)
                    if (dir_cy(i) != 0) {
                        const T v = __ldg(h + (long long)pop_plane(1 - k, i) * NP + zs[1 - dir_cz(i)] + (long long)gy * nx + xs[1 - dir_cx(i)]);
                        if ((dir_cy(i) > 0 && wrap_ylo) || (dir_cy(i) < 0 && wrap_yhi)) fo[i] = v;
                    }
            }
            moments19<T>(fo, orho, ojx, ojy, ojz);
        } else {
            T* mine = st + rd0;
            mine[L::slot_off(0)] = rho; mine[L::slot_off(3)] = jx; mine[L::slot_off(4)] = jy; mine[L::slot_off(5)] = jz;
            asm volatile("bar.sync %0, 64;" ::"r"(ty + 1) : "memory");     // the two warps (red, blue) of this tile row
            const T* other = st + rd0 + (1 - 2 * k) * NT;                  // the partner's entries (other component, same node)
            orho = other[L::slot_off(0)]; ojx = other[L::slot_off(3)]; ojy = other[L::slot_off(4)]; ojz = other[L::slot_off(5)];
        }
        {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy accesses to the stage before the TMA's next writes
            __syncwarp();
            if (lane_lo) mbar_arrive(done + sg);        // the producer may refill this stage with the plane after next
            if (fluid) {
                // common velocity (S4): u' = (om_r j^r + om_b j^b) / (om_r rho^r + om_b rho^b).  Both threads of the node must
                // get the same bits: separately rounded products and one sum are commutative, a contracted fma is not.
                const T om_own = cst[k], om_oth = cst[1 - k];
                const T den = add_rn(mul_rn(om_own, rho), mul_rn(om_oth, orho));
                const T inv = den != zero ? T(1) / den : zero;
                ux = add_rn(mul_rn(om_own, jx), mul_rn(om_oth, ojx)) * inv;
                uy = add_rn(mul_rn(om_own, jy), mul_rn(om_oth, ojy)) * inv;
                uz = add_rn(mul_rn(om_own, jz), mul_rn(om_oth, ojz)) * inv;
            }
        }
        if (fluid) {
            // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6); a solid neighbour counts psi = 0 (S7)
            T d[9];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                T vp = ring_o[sp * 2 * RS + pair_cy(p) * RW + pair_cx(p)];
                T vm = ring_o[sm_ * 2 * RS - pair_cy(p) * RW - pair_cx(p)];
                if (HAS_SOLID) {
                    if (lk >> (2 * p + 1) & 1u) vp = zero;
                    if (lk >> (2 * p + 2) & 1u) vm = zero;
                }
                d[p] = w_pair<T>(p) * (vp - vm);
            }
            const T gx = (((d[0] + d[3]) + d[4]) + d[5]) + d[6];
            const T gy = (((d[1] + d[3]) - d[4]) + d[7]) + d[8];
            const T gz = (((d[2] + d[5]) - d[6]) + d[7]) - d[8];
            const T G_ = cst[2];
            ex = ux - G_ * gx; ey = uy - G_ * gy; ez = uz - G_ * gz;
        }
        }   // MODEL == 0
        if (DIAG) {
            const double om = 1.0 - double(omc), r_ = store_h ? double(rho) : 0.0;      // the re-collided planes belong to another chunk
            double v0 = r_, v1 = r_ == 0.0 ? 0.0 : double(omc) * double(jx) + r_ * (om * double(ux) + (double(ex) - double(ux)));
            double v2 = r_ == 0.0 ? 0.0 : double(omc) * double(jy) + r_ * (om * double(uy) + (double(ey) - double(uy)));
            double v3 = r_ == 0.0 ? 0.0 : double(omc) * double(jz) + r_ * (om * double(uz) + (double(ez) - double(uz)));
            // four values, 32 lanes: two halving steps, then three plain ones; lanes 0, 8, 16, 24 end up with the sums of v0, v1, v2, v3
            const bool hA = (tx & 16) != 0, hB = (tx & 8) != 0;
            double kA = hA ? v2 : v0, kB = hA ? v3 : v1;
            kA += __shfl_xor_sync(0xffffffffu, hA ? v0 : v2, 16);
            kB += __shfl_xor_sync(0xffffffffu, hA ? v1 : v3, 16);
            double kk_ = hB ? kB : kA;
            kk_ += __shfl_xor_sync(0xffffffffu, hB ? kA : kB, 8);
            kk_ += __shfl_xor_sync(0xffffffffu, kk_, 4);
            kk_ += __shfl_xor_sync(0xffffffffu, kk_, 2);
            kk_ += __shfl_xor_sync(0xffffffffu, kk_, 1);
            if ((tx & 7) == 0) {
                double* wa = reinterpret_cast<double*>(smem_tma + L::WACC_BYTE_OFF) + (t / 32) * 4 + (hA ? 2 : 0) + (hB ? 1 : 0);
                *wa = (it == 0 ? 0.0 : *wa) + kk_;
            }
        }

        // ---- BGK collision with exact-difference forcing (Eq. 1, Eq. 10, S5), and, pair by pair as the post-collision values
        //      appear: their (aligned, coalesced) stores and the x stage of the density gather
        //      rho(y, t+1) = sum_i h_i(y - c_i): x by warp shuffles, z by register pipelines, y through shared memory.
        //      A solid node runs the same instructions on zeros (the shuffles need every lane) and stores those zeros. ----
        // The row sums go straight into the z pipelines of the gather, one per y class (0: c_y = 0, p: c_y = +1, m: c_y = -1):
        // a* = V_+1(z-2) + V_0(z-1) so far, completed by V_-1(z) for plane z-1; b* = V_+1(z-1), taking V_0(z); c* = V_+1(z).
        T qc0 = zero, qcp = zero, qcm = zero;
        T* SUup = SU;                                    // interior: Up summed over z (plane z-1); x frame: Up[c_z = 0] of the virtual column, plane z
        T* SUum = SU + SUP;
        T bs = zero;                                     // bounced-back arrivals of the next step come from this node
        // Every plane is stored, also the two re-collided ones at the chunk ends (their owner chunk writes the same bits from the
        // same inputs), and with solids every node too: a solid node has collided zeros into zeros, which is what its populations
        // are in both buffers (S8).  A predicate per store cost 7 % on config 4 (partly written sectors), 3 % without solids.
        T* o = g + (e_own + zl * plu);                   // values arrive in direction order: a running pointer, two planes per step
        auto put = [&](T v) {
            st_global(o, v);
            ptr_step16(o, step16);
        };
        auto on_rest = [&](T h0) { put(h0); qb0 += h0; };
        auto on_pair = [&](int p, T h1, T h2) {
                put(h1);
                put(h2);
                if (HAS_SOLID) {
                    if (lk >> (2 * p + 1) & 1u) bs += h1;
                    if (lk >> (2 * p + 2) & 1u) bs += h2;
                }
                T l = zero, r = zero;
                if (p == 0 || (p >= 3 && p <= 6)) { l = __shfl_up_sync(0xffffffffu, h1, 1); r = __shfl_down_sync(0xffffffffu, h2, 1); }
                if (p == 0) {                                              // +x / -x
                    if (!lane_lo) qb0 += l;
                    if (!lane_hi) qb0 += r;
                    if (lane_hi) exs[1] = h1;                              // what leaves the tile in x with c_y = 0, by c_z
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
                    const bool main_diag = lane_hi == row_hi;              // (hi, hi) and (lo, lo) export along +x+y / -x-y (p = 3), the others along +x-y / -x+y (p = 4)
                    if ((p == 3) == main_diag) {
                        // (hi, hi) +x+y -> entry 0 of tile (y+, x+); (lo, lo) -x-y -> 3 of (y-, x-); (hi, lo) +x-y -> 2 of (y-, x+); (lo, hi) -x+y -> 1 of (y+, x-)
                        const int kk = opaque(k);
                        const unsigned e_xy = unsigned(kk * ro.s_xy) + ((row_hi ? btyp : btym) * ntx + (lane_hi ? btxp : btxm)) * 4 + (row_hi ? (lane_hi ? 0 : 1) : (lane_hi ? 2 : 3));
                        ro.xy[e_xy + zl * psxy] = lane_hi ? h1 : h2;
                    }
                }
            };
        if constexpr (MODEL == 0) collide19_pairs<T>(f, rho, omc, ux, uy, uz, ex, ey, ez, on_rest, on_pair);
        else collide19_cg_pairs<T>(f, cg_rt, cg_x, cg_om, ux, uy, uz, cg_amp, ex, ey, ez, cg_ig2, cg_ign, cg_rcs, on_rest, on_pair);
        if (HAS_SOLID) qb0 += bs;
        // the collision was the last reader of this plane's link word: fetch the next plane's here, so that its latency
        // hides behind the rest of the iteration (at the end of the iteration instead: config 4 2.36 -> 2.27 ms)
        if (HAS_SOLID && it + 1 < NITER()) lk = __ldg(links + (e_own - unsigned(k * NP)) + (long long)(zl + 1 == nz ? 0 : zl + 1) * pl);
        const T p0 = qa0, pp = qap, pm = qam;               // complete for plane z-1
        qa0 = qb0; qb0 = qc0;
        qap = qbp; qbp = qcp;
        qam = qbm; qbm = qcm;
        SUup[0] = pp;
        SUum[0] = pm;
        __syncwarp();
        if (lane_lo) mbar_arrive(rowpub + sg * 2 * TY + k * TY + ty);

        // ---- global stores that need nothing from the other warps: the y-edge exports ----
        if ((row_lo || row_hi) && store_rho) {                             // the row beyond the tile edge receives exactly Um (Up)
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

        // ---- y stage of the gather; exports across the tile's x edges ----
        {
            T out = p0;
            if (!row_lo) out += SUup[-RW];                                 // Up(y-1)
            if (!row_hi) out += SUum[RW];                                  // Um(y+1)
            if (store_rho) ro.in[e_own + zt * plu] = out;
            if (lane_lo || lane_hi) {
                const int vc = lane_lo ? -1 : 1;                           // the virtual column next to this lane
                T a_0 = exs[1];
                if (!row_lo) a_0 += SUup[vc - RW];
                if (!row_hi) a_0 += SUum[vc + RW];
                const T hout = exs[3] + exs[0];                            // z pipeline of the export, as above
                exs[3] = exs[4] + a_0;
                exs[4] = exs[2];
                if (store_rho) {
                    const int kk = opaque(k);
                    const unsigned e_x = unsigned(kk * ro.s_x) + ((bty * ntx + (lane_lo ? btxm : btxp)) * 2 + (lane_lo ? 1 : 0)) * TY + ty;
                    ro.x[e_x + zt * psx] = hout;
                }
            }
        }
        zt = zl;
        zl = zl + 1 == nz ? 0 : zl + 1;
    }
    if (DIAG) {
        asm volatile("bar.sync 9, %0;" ::"n"(NC) : "memory");              // every consumer warp's sums are in place
        if (t < 5) {
            const double* wp = reinterpret_cast<const double*>(smem_tma + L::WACC_BYTE_OFF);
            double s = 0.0;
            if (t < 2) { for (int w = 0; w < TY; ++w) s += wp[(t * TY + w) * 4]; }
            else { for (int w = 0; w < 2 * TY; ++w) s += wp[w * 4 + t - 1]; }
            const long long cta = blockIdx.x + (long long)gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z);
            diag_part[cta * 5 + t] = s;
        }
    }
}

}  // namespace lb
